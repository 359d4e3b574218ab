// k_z<48> and k_zm<48> (see pgsf_zpass.cuh)
#include "pgsf_zpass.cuh"

PGSF_INSTANTIATE_Z(48)
