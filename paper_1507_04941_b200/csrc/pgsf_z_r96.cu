// k_z<96> and k_zm<96> (see pgsf_zpass.cuh)
#include "pgsf_zpass.cuh"

PGSF_INSTANTIATE_Z(96)
