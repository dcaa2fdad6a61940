// TMA-staged kernels for neighbour-list row width K = 3 (see kg_staged_impl.cuh).
#define KG_STAGED_K 3
#include "kg_staged_impl.cuh"
