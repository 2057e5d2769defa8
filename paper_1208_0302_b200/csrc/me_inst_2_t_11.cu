// Specialisation: 2 line(s), effective triplets, 11 parameters.
#define ME_INST_NL 2
#define ME_INST_TRIPLET true
#define ME_INST_TAG t
#define ME_INST_M 11
#include "me_inst.cuh"
