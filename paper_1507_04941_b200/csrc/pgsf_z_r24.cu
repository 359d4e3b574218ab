// k_z<24> and k_zm<24> (see pgsf_zpass.cuh)
#include "pgsf_zpass.cuh"

PGSF_INSTANTIATE_Z(24)
