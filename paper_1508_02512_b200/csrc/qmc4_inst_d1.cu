#include "qmc_inst4.cuh"
QMC4_DEFINE_DIM(1)
