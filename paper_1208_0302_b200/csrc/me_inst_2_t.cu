// Specialisation: 2 line(s), effective triplets.
#define ME_INST_NL 2
#define ME_INST_TRIPLET true
#define ME_INST_TAG t
#include "me_inst.cuh"
