// k_prox_res_10.cu - k_prox_res<LOTS = 1, CHECK = 0> (see k_prox_res_inst.inc)
#define RES_LOTS true
#define RES_CHECK false
#define RES_FN(name) prox_res_##name##_10
#include "k_prox_res_inst.inc"
