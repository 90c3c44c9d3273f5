// k_prox_res_01.cu - k_prox_res<LOTS = 0, CHECK = 1> (see k_prox_res_inst.inc)
#define RES_LOTS false
#define RES_CHECK true
#define RES_FN(name) prox_res_##name##_01
#include "k_prox_res_inst.inc"
