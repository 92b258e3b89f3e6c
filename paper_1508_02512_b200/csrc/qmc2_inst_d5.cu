#include "qmc_inst2.cuh"
QMC2_DEFINE_DIM(5)
