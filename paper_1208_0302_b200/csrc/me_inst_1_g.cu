// Specialisation: 1 line(s), general Zeeman component lists.
#define ME_INST_NL 1
#define ME_INST_TRIPLET false
#define ME_INST_TAG g
#include "me_inst.cuh"
