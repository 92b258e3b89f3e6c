#include "qmc_inst.cuh"
QMC_DEFINE_DIM(5)
