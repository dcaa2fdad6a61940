// TMA-staged kernels for neighbour-list row width K = 9 (next-nearest-neighbour honeycomb; see kg_staged_impl.cuh).
#define KG_STAGED_K 9
#include "kg_staged_impl.cuh"
