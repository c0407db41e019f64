// chem_tps_inst_a.cu -- compile-time-N instantiations of the thread-per-state kernel (chem_tps_kernel.cuh), N = 8..12
#include "chem_tps_kernel.cuh"
CHEM_TPS_INSTANTIATE(8)
CHEM_TPS_INSTANTIATE(9)
CHEM_TPS_INSTANTIATE(10)
CHEM_TPS_INSTANTIATE(11)
CHEM_TPS_INSTANTIATE(12)
