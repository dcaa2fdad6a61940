// TMA-staged kernels for neighbour-list row width K = 6 (see kg_staged_impl.cuh).
#define KG_STAGED_K 6
#include "kg_staged_impl.cuh"
