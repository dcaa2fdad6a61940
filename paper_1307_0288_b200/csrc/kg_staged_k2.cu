// TMA-staged kernels for neighbour-list row width K = 2 (see kg_staged_impl.cuh).
#define KG_STAGED_K 2
#include "kg_staged_impl.cuh"
