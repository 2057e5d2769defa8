// Specialisation: up to 4 (run-time) line(s), general component lists, 9 parameters.
#define ME_INST_NL 4
#define ME_INST_TRIPLET false
#define ME_INST_TAG g
#define ME_INST_M 9
#include "me_inst.cuh"
