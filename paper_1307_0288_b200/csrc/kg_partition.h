// kg_partition.h — host side of the site re-ordering done at create.
//
// The Chebyshev moments of Alg. 5 are inner products, so they do not depend on the order
// in which the sites are numbered; the kernels do: a tile of consecutive sites is staged in shared
// memory, and every bond that leaves the tile costs a gather through L2 (kg_staged.cuh) or a halo
// site that has to be brought in and recomputed (kg_tb2.cuh).  With the caller's numbering — e.g. the
// row-major cells of a 1000 x 1000-cell sheet — a tile is a one-cell-high strip and nearly every
// site has a bond that leaves it.  kg_partition renumbers the sites so that every aligned range of
// leaf * 2^j consecutive sites is a compact patch of the lattice.
//
// Method: recursive graph bisection along breadth-first level structures (George & Liu's level
// structures; "recursive graph bisection" of the mesh-partitioning literature), using only the
// neighbour list: a set of sites is ordered breadth-first from a peripheral site, the first part of
// that order (a whole number of leaves, the largest power of two below the leaf count — so that
// every power-of-two block starts aligned) becomes the left child, the rest the right child; the
// left child is re-ordered from the same start site, the right child from the site visited last (the
// far end).  Inside a leaf the sites keep the caller's relative order.  Cost O(n K log(n / leaf)); no coordinates are
// needed, so it works for every list kg_create_hamiltonian[_csr] accepts (sheets, ribbons, vacancies,
// cubic lattices, ...).  Plain host C++, no CUDA.
#pragma once
#include <stdint.h>

#include <algorithm>
#include <vector>

// perm[new] = old.  nl is the k-major list of kg_create_hamiltonian (nl[k*n + i], k < nn[i]).
// Entries outside [0, n) or k >= kmax are ignored here (create validates them on the device).
static inline void kg_partition_host(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, int64_t leaf,
                                     std::vector<int32_t> &perm)
{
    perm.resize((size_t)n);
    if (n <= 0) return;
    if (leaf < 1) leaf = 1;
    std::vector<int32_t> node((size_t)n, 0);      // tree node the site currently belongs to
    std::vector<int32_t> tmp((size_t)n);
    std::vector<uint8_t> seen((size_t)n, 0);
    for (int64_t i = 0; i < n; ++i) perm[(size_t)i] = (int32_t)i;

    struct Seg { int64_t b, e; int32_t start; int32_t id; };
    std::vector<Seg> stack;
    int32_t next_id = 1;
    stack.push_back(Seg{0, n, 0, 0});
    while (!stack.empty()) {
        const Seg sg = stack.back();
        stack.pop_back();
        const int64_t cnt = sg.e - sg.b;
        // breadth-first order of the segment's sites from sg.start (restricted to the segment);
        // components that are not reached are appended in the segment's current order
        int64_t head = sg.b, tail = sg.b;
        auto push = [&](int32_t v) { seen[(size_t)v] = 1; tmp[(size_t)tail++] = v; };
        push(sg.start);
        int64_t scan = sg.b;
        int32_t last = sg.start;
        while (tail < sg.e || head < tail) {
            if (head == tail) {                     // next component
                while (seen[(size_t)perm[(size_t)scan]]) ++scan;
                push(perm[(size_t)scan]);
            }
            const int32_t v = tmp[(size_t)head++];
            last = v;
            int c = nn[v];
            if (c > kmax) c = kmax;
            for (int k = 0; k < c; ++k) {
                const int32_t m = nl[(int64_t)k * n + v];
                if (m < 0 || m >= n || seen[(size_t)m] || node[(size_t)m] != sg.id) continue;
                push(m);
            }
        }
        for (int64_t q = sg.b; q < sg.e; ++q) { perm[(size_t)q] = tmp[(size_t)q]; seen[(size_t)tmp[(size_t)q]] = 0; }
        const int64_t nleaves = (cnt + leaf - 1) / leaf;
        if (nleaves <= 1) {
            // inside a leaf the caller's order is kept: consecutive sites of a lattice row stay consecutive, and
            // so do their neighbours (regular strides: fewer shared-memory bank conflicts in the gathers)
            std::sort(perm.begin() + sg.b, perm.begin() + sg.e);
            continue;
        }
        int64_t lp = 1;
        while (lp * 2 < nleaves) lp *= 2;          // largest power of two below the leaf count
        const int64_t mid = sg.b + lp * leaf;
        const int32_t idl = next_id++, idr = next_id++;
        for (int64_t q = sg.b; q < mid; ++q) node[(size_t)perm[(size_t)q]] = idl;
        for (int64_t q = mid; q < sg.e; ++q) node[(size_t)perm[(size_t)q]] = idr;
        // right child first on the stack so that the left one is processed next (depth-first, left to right)
        int32_t rstart = last;
        if (node[(size_t)rstart] != idr) rstart = perm[(size_t)(sg.e - 1)];
        stack.push_back(Seg{mid, sg.e, rstart, idr});
        stack.push_back(Seg{sg.b, mid, perm[(size_t)sg.b], idl});
    }
}

// The same bisection on GROUPS of `group` consecutive caller sites (group = 8: "octets"), so that an
// internal site keeps its caller index modulo `group`:  internal = 8 * (position of its octet) + caller % 8.
// Why: the kernels gather T_m[neighbour] from a tile staged in shared memory with 16-byte loads, eight
// lanes (= eight consecutive sites) per wavefront; the eight loads are conflict-free when they fall into
// eight different 16-byte bank groups, i.e. when the neighbours' slots differ modulo 8.  In a regularly
// numbered lattice (the paper's row-major honeycomb cells) the k-th neighbours of eight consecutive
// sites have eight different caller indices modulo 8, and an order that preserves the caller index
// modulo 8 carries that over to the slots wherever the octets are placed; a site-by-site re-ordering
// makes the residues random (2.3 wavefronts per gather instead of 1, profiles/r02b_tb2.md).
// The trailing partial group, if any, stays last.  perm[new] = old.
static inline void kg_partition_grouped(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, int64_t leaf, int group,
                                        std::vector<int32_t> &perm)
{
    if (group <= 1 || n < 2 * (int64_t)group) { kg_partition_host(n, kmax, nn, nl, leaf, perm); return; }
    const int64_t ngf = n / group;                 // full groups (a trailing partial group is kept out)
    // quotient graph: groups adjacent when any of their sites are
    std::vector<int32_t> deg((size_t)ngf, 0), adj((size_t)ngf * group * kmax, -1);
    const int64_t stride = (int64_t)group * kmax;
    int kq = 0;
    for (int64_t g = 0; g < ngf; ++g) {
        int32_t *a = adj.data() + (size_t)g * stride;
        int d = 0;
        for (int64_t i = g * group; i < (g + 1) * group; ++i) {
            int c = nn[i];
            if (c > kmax) c = kmax;
            for (int k = 0; k < c; ++k) {
                const int32_t m = nl[(int64_t)k * n + i];
                if (m < 0 || m >= n) continue;
                const int32_t mg = (int32_t)(m / group);
                if (mg == g || mg >= ngf) continue;
                bool seen = false;
                for (int q = 0; q < d; ++q) seen = seen || a[q] == mg;
                if (!seen) a[d++] = mg;
            }
        }
        deg[(size_t)g] = d;
        kq = std::max(kq, d);
    }
    if (kq == 0) kq = 1;
    std::vector<int32_t> nlq((size_t)ngf * kq, 0);
    for (int64_t g = 0; g < ngf; ++g)
        for (int k = 0; k < deg[(size_t)g]; ++k) nlq[(size_t)k * ngf + g] = adj[(size_t)g * stride + k];
    adj.clear(); adj.shrink_to_fit();
    std::vector<int32_t> pq;
    kg_partition_host(ngf, kq, deg.data(), nlq.data(), std::max<int64_t>(1, leaf / group), pq);
    perm.resize((size_t)n);
    int64_t pos = 0;
    for (int64_t g = 0; g < ngf; ++g)
        for (int j = 0; j < group; ++j) perm[(size_t)pos++] = (int32_t)((int64_t)pq[(size_t)g] * group + j);
    for (int64_t i = ngf * group; i < n; ++i) perm[(size_t)pos++] = (int32_t)i;
}
