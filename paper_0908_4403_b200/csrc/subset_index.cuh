// subset_index.cuh -- ranking of photon subsets by size, shared by amp2_subset.cu and
// amp2_twosided.cu (product code).  One copy of the table per translation unit (static
// __constant__), copied to shared memory by the kernels that index it per lane.
#pragma once

constexpr int kMaxN = 8;

__host__ __device__ constexpr int binom(int n, int k)
{
    if (k < 0 || k > n) return 0;
    int r = 1;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}

// rank[S]: position of S among the subsets with the same number of elements, in increasing
// numeric order; list[m][r]: its inverse.  Independent of N for S < 2^N.
struct SubsetIndex {
    unsigned char rank[1 << kMaxN];
    unsigned char list[kMaxN + 1][72];
};

constexpr SubsetIndex make_subset_index()
{
    SubsetIndex t{};
    int count[kMaxN + 1] = {};
    for (int S = 0; S < (1 << kMaxN); ++S) {
        int m = 0;
        for (int b = 0; b < kMaxN; ++b) m += (S >> b) & 1;
        t.rank[S] = (unsigned char)count[m];
        t.list[m][count[m]] = (unsigned char)S;
        ++count[m];
    }
    return t;
}

static __constant__ SubsetIndex c_index = make_subset_index();


// copy the part of the index tables that N photons use into shared memory:
// s_rank[0 .. 2^N), s_list[m * 72 + r] for m <= N, r < C(N, m)   (row stride 72 as in c_index)
template <int N, int THREADS>
__device__ __forceinline__ void load_subset_index(unsigned char* s_rank, unsigned char* s_list)
{
    constexpr int COLS = binom(N, N / 2);  // widest row
    for (int i = threadIdx.x; i < (1 << N); i += THREADS) s_rank[i] = c_index.rank[i];
    for (int i = threadIdx.x; i < (N + 1) * COLS; i += THREADS)
        s_list[(i / COLS) * 72 + i % COLS] = c_index.list[i / COLS][i % COLS];
}
