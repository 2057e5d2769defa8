// Specialisation: 4 line(s) (run-time count up to ME_MAX_LINES), general Zeeman component lists.
#define ME_INST_NL 4
#define ME_INST_TRIPLET false
#define ME_INST_TAG g
#include "me_inst.cuh"
