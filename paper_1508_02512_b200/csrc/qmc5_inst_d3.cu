#include "qmc_inst5.cuh"
QMC5_DEFINE_DIM(3)
