// chem_tps_inst_b.cu -- compile-time-N instantiations of the thread-per-state kernel (chem_tps_kernel.cuh), N = 14..16
#include "chem_tps_kernel.cuh"
CHEM_TPS_INSTANTIATE(14)
CHEM_TPS_INSTANTIATE(15)
CHEM_TPS_INSTANTIATE(16)
