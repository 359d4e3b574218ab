// k_z<6> and k_zm<6> (see pgsf_zpass.cuh)
#include "pgsf_zpass.cuh"

PGSF_INSTANTIATE_Z(6)
