// k_z<72> and k_zm<72> (see pgsf_zpass.cuh)
#include "pgsf_zpass.cuh"

PGSF_INSTANTIATE_Z(72)
