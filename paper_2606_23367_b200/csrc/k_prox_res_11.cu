// k_prox_res_11.cu - k_prox_res<LOTS = 1, CHECK = 1> (see k_prox_res_inst.inc)
#define RES_LOTS true
#define RES_CHECK true
#define RES_FN(name) prox_res_##name##_11
#include "k_prox_res_inst.inc"
