// Test harness for csrc/kg_partition.h (host-only C++): reads a k-major neighbour list, writes perm.
//   partition_cli <n> <kmax> <leaf> <group> <in.bin> <out.bin>
// in.bin = int32 nn[n] followed by int32 nl[kmax*n]; out.bin = int32 perm[n] (perm[new] = old).
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../../paper_1307_0288_b200/csrc/kg_partition.h"

int main(int argc, char **argv)
{
    if (argc != 7) return 2;
    const int64_t n = atoll(argv[1]);
    const int kmax = atoi(argv[2]);
    const int64_t leaf = atoll(argv[3]);
    const int group = atoi(argv[4]);
    std::vector<int32_t> nn((size_t)n), nl((size_t)n * kmax), perm;
    FILE *f = fopen(argv[5], "rb");
    if (!f || fread(nn.data(), 4, (size_t)n, f) != (size_t)n || fread(nl.data(), 4, (size_t)n * kmax, f) != (size_t)n * kmax) return 3;
    fclose(f);
    if (group > 1) kg_partition_grouped(n, kmax, nn.data(), nl.data(), leaf, group, perm);
    else kg_partition_host(n, kmax, nn.data(), nl.data(), leaf, perm);
    f = fopen(argv[6], "wb");
    if (!f || fwrite(perm.data(), 4, (size_t)n, f) != (size_t)n) return 4;
    fclose(f);
    return 0;
}
