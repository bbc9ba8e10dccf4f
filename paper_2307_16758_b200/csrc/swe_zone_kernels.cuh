// swe_zone_kernels.cuh -- ghost-layer generation on the device (
// PAPER.md:86-127, section 3.2 "Adding layers of ghost cells" and 3.3 "Renumbering the cells").
//
// The paper finds the ghost cells of a sub-domain by exchanging bounding boxes and inner boundary
// layers between MPI ranks and then following the connectivity layer by layer.  With the whole
// mesh resident in one GPU's HBM neither exchange is needed: the k layers of ALL zones grow
// together, one wavefront step per layer, as bit masks over the edge adjacency:
//
//   reach_0[c]   = { zone_of[c] }                                   (one bit per zone)
//   reach_l[c]   = reach_{l-1}[c]  |  OR_k reach_{l-1}[nb_k(c)]      (three gathers per cell)
//   fresh_l[c]   = reach_l[c] & ~reach_{l-1}[c]   = the zones that get c as a layer-l ghost
//
// (breadth-first distance over the edge adjacency, A.12.2).  Every set bit becomes one 64-bit key
//   ((z * nz + src) * 4 + l) << 32 | c ,   src = zone_of[c],
// and a least-significant-digit radix sort of the keys gives the numbering of section 3.3: per
// zone z the ghosts grouped by source zone (one contiguous receive range per neighbour), inside a
// group by layer and then by cell id (A.12.3).  Set-up code: runs once per swe_zones_create.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace swe {

// masks are stored word-major: word w of cell c at mask[w * nc + c]; W = ceil(nz / 64) words
__global__ void __launch_bounds__(256) k_gl_seed(const int* __restrict__ zone_of, unsigned long long* __restrict__ reach,
                                                 int nc, int W) {
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        const int z = zone_of[c];
        for (int w = 0; w < W; ++w) reach[(size_t)w * nc + c] = ((z >> 6) == w) ? (1ull << (z & 63)) : 0ull;
    }
}

// one layer: nxt = cur | cur[neighbours], fresh = nxt & ~cur; *count += number of set bits in fresh
__global__ void __launch_bounds__(256) k_gl_grow(const int4* __restrict__ c2c, const unsigned long long* __restrict__ cur,
                                                 unsigned long long* __restrict__ nxt, unsigned long long* __restrict__ fresh,
                                                 int nc, int W, unsigned long long* count) {
    unsigned int local = 0;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        const int4 nb = c2c[c];
        for (int w = 0; w < W; ++w) {
            const unsigned long long* m = cur + (size_t)w * nc;
            const unsigned long long own = m[c];
            unsigned long long r = own;
            if (nb.x >= 0) r |= m[nb.x];
            if (nb.y >= 0) r |= m[nb.y];
            if (nb.z >= 0) r |= m[nb.z];
            const unsigned long long f = r & ~own;
            nxt[(size_t)w * nc + c] = r;
            fresh[(size_t)w * nc + c] = f;
            local += __popcll(f);
        }
    }
    for (int o = 16; o > 0; o >>= 1) local += __shfl_down_sync(0xffffffffu, local, o);
    if ((threadIdx.x & 31) == 0 && local) atomicAdd(count, (unsigned long long)local);
}

// one key per set bit of fresh (any order: the sort that follows covers every key bit)
__global__ void __launch_bounds__(256) k_gl_emit(const unsigned long long* __restrict__ fresh, const int* __restrict__ zone_of,
                                                 int layer, int nz, int nc, int W, unsigned long long* __restrict__ keys,
                                                 unsigned long long* cursor) {
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        for (int w = 0; w < W; ++w) {
            unsigned long long f = fresh[(size_t)w * nc + c];
            if (!f) continue;
            const unsigned long long src = (unsigned long long)zone_of[c];
            const unsigned long long at = atomicAdd(cursor, (unsigned long long)__popcll(f));
            int j = 0;
            while (f) {
                const int b = __ffsll((long long)f) - 1;
                f &= f - 1;
                const unsigned long long z = (unsigned long long)(w * 64 + b);
                keys[at + j++] = (((z * nz + src) * 4ull + (unsigned long long)layer) << 32) | (unsigned int)c;
            }
        }
    }
}

// ---- stable least-significant-digit radix sort of 64-bit keys, 8 bits per pass ----
constexpr int RS_THREADS = 256;
constexpr int RS_TILE = 4096;         // keys per block and pass

// hist[d * nblk + blk] = number of keys of block blk's tile with digit d
__global__ void __launch_bounds__(RS_THREADS) k_rs_hist(const unsigned long long* __restrict__ keys, long long n, int shift,
                                                        unsigned int* __restrict__ hist, int nblk) {
    __shared__ unsigned int cnt[256];
    cnt[threadIdx.x] = 0;
    __syncthreads();
    const long long t0 = (long long)blockIdx.x * RS_TILE;
    for (int j = threadIdx.x; j < RS_TILE; j += RS_THREADS) {
        const long long i = t0 + j;
        if (i < n) atomicAdd(&cnt[(unsigned int)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nblk + blockIdx.x] = cnt[threadIdx.x];
}

// exclusive prefix sum of hist[0..m) in place, one block
__global__ void __launch_bounds__(1024) k_rs_scan(unsigned int* __restrict__ hist, long long m) {
    __shared__ unsigned int part[1024];
    const long long per = (m + 1023) / 1024;
    const long long a = per * threadIdx.x, b = (a + per < m) ? a + per : m;
    unsigned int s = 0;
    for (long long i = a; i < b; ++i) s += hist[i];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int run = 0;
        for (int i = 0; i < 1024; ++i) { const unsigned int v = part[i]; part[i] = run; run += v; }
    }
    __syncthreads();
    unsigned int run = part[threadIdx.x];
    for (long long i = a; i < b; ++i) { const unsigned int v = hist[i]; hist[i] = run; run += v; }
}

// stable scatter: the tile is walked in rounds of 256 consecutive keys; inside a round the rank of
// a key among the equal digits before it comes from __match_any_sync (within the warp) and the
// per-warp digit counts (across the warps of the block)
// VAL: a 32-bit value travels with every key (vin -> vout)
template <bool VAL>
__global__ void __launch_bounds__(RS_THREADS) k_rs_scatter(const unsigned long long* __restrict__ in,
                                                           unsigned long long* __restrict__ out, long long n, int shift,
                                                           const unsigned int* __restrict__ hist, int nblk,
                                                           const unsigned int* __restrict__ vin = nullptr,
                                                           unsigned int* __restrict__ vout = nullptr) {
    __shared__ unsigned int base[256];
    __shared__ unsigned int wcnt[RS_THREADS / 32][256];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    base[tid] = hist[(size_t)tid * nblk + blockIdx.x];
    #pragma unroll
    for (int w = 0; w < RS_THREADS / 32; ++w) wcnt[w][tid] = 0;
    __syncthreads();
    const long long t0 = (long long)blockIdx.x * RS_TILE;
    for (int r = 0; r < RS_TILE / RS_THREADS; ++r) {
        const long long i = t0 + (long long)r * RS_THREADS + tid;
        const bool valid = i < n;
        const unsigned long long key = valid ? in[i] : 0ull;
        const unsigned int d = valid ? ((unsigned int)(key >> shift) & 255u) : 256u;
        const unsigned int peers = __match_any_sync(0xffffffffu, d);
        const unsigned int rank = __popc(peers & ((1u << lane) - 1u));
        if (valid && rank == 0) wcnt[wid][d] = __popc(peers);
        __syncthreads();
        if (valid) {
            unsigned int off = base[d] + rank;
            for (int w = 0; w < wid; ++w) off += wcnt[w][d];
            out[off] = key;
            if (VAL) vout[off] = vin[i];
        }
        __syncthreads();
        unsigned int tot = 0;
        #pragma unroll
        for (int w = 0; w < RS_THREADS / 32; ++w) { tot += wcnt[w][tid]; wcnt[w][tid] = 0; }
        base[tid] += tot;
        __syncthreads();
    }
}

}  // namespace swe
