// Allen-Cahn 2D (kind 3) product-form projection kernel (in-SMEM level solves).
#include "kernels_2d_direct.cuh"
