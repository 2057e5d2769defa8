// Specialisation: 4 line(s) (run-time count up to ME_MAX_LINES), effective triplets.
#define ME_INST_NL 4
#define ME_INST_TRIPLET true
#define ME_INST_TAG t
#include "me_inst.cuh"
