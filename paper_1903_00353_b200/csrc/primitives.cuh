// primitives.cuh -- hand-written device-wide exclusive scan and stable LSD radix sort.
// (The paper calls thrust::sort_by_key / gather; these replace them.)
#pragma once
#include "common.cuh"

// =========================================================================================
// exclusive scan: three phases (tile reduce -> single-block scan of tile sums -> tile scan)
//   InF  : u64 operator()(int64_t i)                      value of element i
//   OutF : void operator()(int64_t i, u64 excl, u64 v)    consume exclusive prefix of element i
// Tile = SCAN_BT threads x SCAN_IPT consecutive elements per thread.
// =========================================================================================
#define SCAN_BT 256
#define SCAN_IPT 8
#define SCAN_TILE (SCAN_BT * SCAN_IPT)

__device__ __forceinline__ u64 warp_incl_scan(u64 v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u64 t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

// block-wide exclusive scan of one value per thread; returns exclusive prefix, total in *total
__device__ __forceinline__ u64 block_excl_scan(u64 v, u64 *total) {
    __shared__ u64 s_w[SCAN_BT / 32];
    __shared__ u64 s_tot;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    u64 inc = warp_incl_scan(v, lane);
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    if (w == 0) {
        u64 x = (lane < SCAN_BT / 32) ? s_w[lane] : 0;
        u64 xi = warp_incl_scan(x, lane);
        if (lane < SCAN_BT / 32) s_w[lane] = xi - x;
        if (lane == SCAN_BT / 32 - 1) s_tot = xi;
    }
    __syncthreads();
    u64 r = s_w[w] + inc - v;
    *total = s_tot;
    __syncthreads();
    return r;
}

template <class InF>
__global__ void __launch_bounds__(SCAN_BT) scan_reduce_kernel(InF in, int64_t n, u64 *partial) {
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_IPT;
    u64 s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_IPT; i++)
        if (base + i < n) s += in(base + i);
    u64 tot;
    block_excl_scan(s, &tot);
    if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

// one block: exclusive scan of partial[0..np) in place, grand total to *total; a thread takes
// SCAN_IPT consecutive values per round
static __global__ void __launch_bounds__(SCAN_BT) scan_partials_kernel(u64 *partial, int64_t np, u64 *total) {
    __shared__ u64 s_run;
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    for (int64_t base = 0; base < np; base += SCAN_TILE) {
        const int64_t i0 = base + (int64_t)threadIdx.x * SCAN_IPT;
        u64 v[SCAN_IPT], s = 0;
#pragma unroll
        for (int k = 0; k < SCAN_IPT; k++) {
            v[k] = (i0 + k < np) ? partial[i0 + k] : 0;
            s += v[k];
        }
        u64 tot;
        u64 ex = block_excl_scan(s, &tot) + s_run;
#pragma unroll
        for (int k = 0; k < SCAN_IPT; k++) {
            if (i0 + k < np) partial[i0 + k] = ex;
            ex += v[k];
        }
        __syncthreads();
        if (threadIdx.x == 0) s_run += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0 && total) *total = s_run;
}

template <class InF, class OutF>
__global__ void __launch_bounds__(SCAN_BT) scan_down_kernel(InF in, OutF out, int64_t n, const u64 *partial) {
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_IPT;
    u64 v[SCAN_IPT];
    u64 s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_IPT; i++) {
        v[i] = (base + i < n) ? in(base + i) : 0;
        s += v[i];
    }
    u64 tot;
    u64 ex = block_excl_scan(s, &tot) + partial[blockIdx.x];
#pragma unroll
    for (int i = 0; i < SCAN_IPT; i++) {
        if (base + i < n) out(base + i, ex, v[i]);
        ex += v[i];
    }
}

static inline size_t scan_ws_elems(int64_t n) { return (size_t)((n + SCAN_TILE - 1) / SCAN_TILE) + 1; }

// ws: at least scan_ws_elems(n) u64; total (device, may be null) receives the grand total.
// inr feeds the reduce pass and ind the down pass: they must return the same values (inr may
// compute and store what ind then only reads back).
template <class InR, class InD, class OutF>
static int launch_scan2(InR inr, InD ind, OutF out, int64_t n, u64 *ws, u64 *total, cudaStream_t st) {
    if (n <= 0) {
        if (total) CK(cudaMemsetAsync(total, 0, sizeof(u64), st));
        return SDF_OK;
    }
    int64_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    KL; scan_reduce_kernel<InR><<<(unsigned)nb, SCAN_BT, 0, st>>>(inr, n, ws);
    KL; scan_partials_kernel<<<1, SCAN_BT, 0, st>>>(ws, nb, total);
    KL; scan_down_kernel<InD, OutF><<<(unsigned)nb, SCAN_BT, 0, st>>>(ind, out, n, ws);
    CK(cudaGetLastError());
    return SDF_OK;
}
template <class InF, class OutF>
static int launch_scan(InF in, OutF out, int64_t n, u64 *ws, u64 *total, cudaStream_t st) {
    return launch_scan2(in, in, out, n, ws, total, st);
}

// =========================================================================================
// stable LSD radix sort, 8-bit digits, key (u32 or u64) + u32 payload
// per pass: tile histograms -> scan (digit-major) -> stable scatter
// =========================================================================================
#define RS_BT 256
#define RS_IPT 8
#define RS_TILE (RS_BT * RS_IPT)
#define RS_WARPS (RS_BT / 32)

template <typename K>
__global__ void __launch_bounds__(RS_BT) radix_hist_kernel(const K *__restrict__ keys, int n, int shift,
                                                           u32 *__restrict__ hist, int nblocks) {
    __shared__ u32 s_h[256];
    s_h[threadIdx.x] = 0;
    __syncthreads();
    int base = blockIdx.x * RS_TILE;
#pragma unroll
    for (int r = 0; r < RS_IPT; r++) {
        int i = base + r * RS_BT + threadIdx.x;
        if (i < n) atomicAdd(&s_h[(u32)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = s_h[threadIdx.x];
}

struct HistIn {
    const u32 *h;
    __device__ u64 operator()(int64_t i) const { return h[i]; }
};
struct HistOut {
    u32 *h;
    __device__ void operator()(int64_t i, u64 ex, u64) const { h[i] = (u32)ex; }
};

template <typename K>
__global__ void __launch_bounds__(RS_BT) radix_scatter_kernel(const K *__restrict__ kin, const u32 *__restrict__ vin,
                                                              K *__restrict__ kout, u32 *__restrict__ vout, int n,
                                                              int shift, const u32 *__restrict__ gofs, int nblocks) {
    __shared__ u32 s_cnt[RS_WARPS][256];
    __shared__ u32 s_base[256];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
#pragma unroll
    for (int i = 0; i < RS_WARPS; i++) s_cnt[i][tid] = 0;
    __syncthreads();
    // warp w owns the contiguous chunk [base, base + 32*RS_IPT) of the tile; round r takes
    // 32 consecutive elements, so (warp, round, lane) order == input order (stability)
    const int base = blockIdx.x * RS_TILE + w * (32 * RS_IPT);
    K key[RS_IPT];
    u32 rank[RS_IPT];
#pragma unroll
    for (int r = 0; r < RS_IPT; r++) {
        int i = base + r * 32 + lane;
        bool valid = i < n;
        key[r] = valid ? kin[i] : (K)0;
        int digit = valid ? (int)((u32)(key[r] >> shift) & 255u) : 256;
        unsigned peers = __match_any_sync(0xffffffffu, digit);
        int leader = __ffs(peers) - 1;
        u32 prev = 0;
        if (lane == leader && valid) {
            prev = s_cnt[w][digit];
            s_cnt[w][digit] = prev + __popc(peers);
        }
        prev = __shfl_sync(0xffffffffu, prev, leader);
        rank[r] = prev + __popc(peers & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    {   // digit tid: exclusive scan of its counts across the warps, plus the global offset
        u32 run = 0;
#pragma unroll
        for (int i = 0; i < RS_WARPS; i++) {
            u32 c = s_cnt[i][tid];
            s_cnt[i][tid] = run;
            run += c;
        }
        s_base[tid] = gofs[(size_t)tid * nblocks + blockIdx.x];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < RS_IPT; r++) {
        int i = base + r * 32 + lane;
        if (i < n) {
            u32 digit = (u32)(key[r] >> shift) & 255u;
            u32 pos = s_base[digit] + s_cnt[w][digit] + rank[r];
            kout[pos] = key[r];
            vout[pos] = vin[i];
        }
    }
}

static inline int radix_blocks(int n) { return (n + RS_TILE - 1) / RS_TILE; }
// u32 words needed for the histogram of one pass
static inline size_t radix_hist_elems(int n) { return (size_t)radix_blocks(n) * 256; }

// Sorts (k0,v0) using (k1,v1) as ping-pong buffers over the digit positions listed in
// shifts[0..npass).  Returns in *result_in_first whether the sorted data ended in (k0,v0).
template <typename K>
static int radix_sort_pairs(K *k0, u32 *v0, K *k1, u32 *v1, int n, const int *shifts, int npass, u32 *hist,
                            u64 *scan_ws, cudaStream_t st, bool *result_in_first) {
    int nb = radix_blocks(n);
    K *ki = k0, *ko = k1;
    u32 *vi = v0, *vo = v1;
    for (int p = 0; p < npass; p++) {
        KL; radix_hist_kernel<K><<<nb, RS_BT, 0, st>>>(ki, n, shifts[p], hist, nb);
        HistIn hin{hist};
        HistOut hout{hist};
        CKS(launch_scan(hin, hout, (int64_t)nb * 256, scan_ws, (u64 *)nullptr, st));
        KL; radix_scatter_kernel<K><<<nb, RS_BT, 0, st>>>(ki, vi, ko, vo, n, shifts[p], hist, nb);
        K *tk = ki; ki = ko; ko = tk;
        u32 *tv = vi; vi = vo; vo = tv;
    }
    CK(cudaGetLastError());
    *result_in_first = (ki == k0);
    return SDF_OK;
}
