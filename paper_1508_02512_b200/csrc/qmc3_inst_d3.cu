#include "qmc_inst3.cuh"
QMC3_DEFINE_DIM(3)
