// k_prox_res_00.cu - k_prox_res<LOTS = 0, CHECK = 0> (see k_prox_res_inst.inc)
#define RES_LOTS false
#define RES_CHECK false
#define RES_FN(name) prox_res_##name##_00
#include "k_prox_res_inst.inc"
