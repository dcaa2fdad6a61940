// TMA-staged kernels for neighbour-list row width K = 4 (see kg_staged_impl.cuh).
#define KG_STAGED_K 4
#include "kg_staged_impl.cuh"
