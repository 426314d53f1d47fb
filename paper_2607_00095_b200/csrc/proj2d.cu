// Allen-Cahn 2D (kind 3) PCG projection kernel.
#include "kernels_2d.cuh"
