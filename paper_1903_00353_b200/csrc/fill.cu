// fill.cu -- sdf_fill_interior: PAPER.md:493 (sec.11.3) "sweeping along
// each of the coordinate axes and filling in unset values in the interior of the geometry", which
// removes the secondary zero crossing between the negative limit of the narrow band and the unset
// interior.  Walking a grid line keeps the sign of the last set cell; an unset (+inf) cell met
// while that sign is negative is set to -band.  Axes x, y, z in turn, every line forward and then
// backward, in place, cells set by an earlier walk counting as set -- the order in which the
// oracle (oracle_fill_interior) does it, so the result is identical cell for cell.
//
// HBM-bound: 4 B per cell read per sweep, the interior written once.
#include "common.cuh"
#include <math.h>
#include <stdlib.h>

// ---- x: one warp per row; a chunk of 32 cells is resolved with two ballots
__device__ __forceinline__ int state_from_left(unsigned set, unsigned neg, int lane, int carry) {
    const unsigned m = set & (0xFFFFFFFFu >> (31 - lane));        // set cells at or before this lane
    if (!m) return carry;
    const int b = 31 - __clz(m);
    return ((neg >> b) & 1u) ? -1 : 1;
}
__device__ __forceinline__ int state_from_right(unsigned set, unsigned neg, int lane, int carry) {
    const unsigned m = set & (0xFFFFFFFFu << lane);               // set cells at or after this lane
    if (!m) return carry;
    const int b = __ffs(m) - 1;
    return ((neg >> b) & 1u) ? -1 : 1;
}

#define SX_BATCH 4       // chunks of 32 cells loaded before they are resolved (memory-level parallelism)
// One walk per row (see sweep_line_kernel for why one is enough).  A chunk of 32 cells is resolved
// with two ballots: an unset cell is filled if the nearest set cell to its left (in the chunk, else
// the carry) or to its right IN THE CHUNK is negative; unset cells with no set cell to their right
// in the chunk join the pending run, which the first set cell of a later chunk resolves (the warp
// then fills the earlier chunks' part of the run with coalesced stores).
//
// Blank map: the walk also records which 32-cell segments of its row are still entirely unset when it
// is done (bit s of word w of the row = segment 32 w + s), once in the order of the y walk and once in
// the order of the z walk.  Most of a grid is such segments -- everything
// outside the band on the outside -- and the y and z walks need not read them (sweep_line_kernel).
__device__ __forceinline__ unsigned chunk_mask(int lane, int a, int b) {      // bits of chunks [a, b) in word `lane`
    const int lo = max(a, 32 * lane), hi = min(b, 32 * lane + 32);
    return lo < hi ? (0xFFFFFFFFu >> (32 - (hi - lo))) << (lo - 32 * lane) : 0u;
}

__global__ void __launch_bounds__(256, 8) sweep_x_kernel(float *__restrict__ dist, int nx, int64_t nrows, float fillv,
                                                      unsigned *__restrict__ blank_y, unsigned *__restrict__ blank_z,
                                                      int nwords, int ny, int nz) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (row >= nrows) return;
    float *d = dist + row * nx;
    int carry = 0, run = -1;
    unsigned bits = 0;           // lane l: word l of the row's blank map
    const bool vec = (nx & 3) == 0 && (((size_t)dist) & 15) == 0;      // every row starts on 16 bytes
    for (int base = 0; base < nx; base += 32 * SX_BATCH) {
        if (vec && base + 32 * SX_BATCH <= nx) {
            // a whole batch without a set cell (most of a grid) is settled from one 128-bit load per lane;
            // otherwise the cells are loaded again the way the chunk logic wants them (from L1)
            static_assert(SX_BATCH == 4, "one float4 per lane covers the batch");
            float4 *qp = reinterpret_cast<float4 *>(d + base) + lane;
            const float4 q = *qp;
            const bool any = isfinite(q.x) || isfinite(q.y) || isfinite(q.z) || isfinite(q.w);
            if (!__any_sync(0xffffffffu, any)) {
                if (carry < 0) {
                    *qp = make_float4(fillv, fillv, fillv, fillv);
                } else {
                    if (run < 0) run = base;
                    if (lane == (base >> 10)) bits |= 0xFu << ((base >> 5) & 31);
                }
                continue;
            }
        }
        float v[SX_BATCH];
#pragma unroll
        for (int u = 0; u < SX_BATCH; u++) {
            const int i = base + 32 * u + lane;
            v[u] = i < nx ? d[i] : INFINITY;
        }
        // a whole batch without a set cell (most of a grid) is settled at once
        bool any = false;
#pragma unroll
        for (int u = 0; u < SX_BATCH; u++) any |= isfinite(v[u]);
        if (!__any_sync(0xffffffffu, any)) {
            const int nch = min(SX_BATCH, (nx - base + 31) >> 5), c0 = base >> 5;      // c0 is a multiple of SX_BATCH
            if (carry < 0) {
                for (int u = 0; u < nch; u++)
                    if (base + 32 * u + lane < nx) d[base + 32 * u + lane] = fillv;
            } else {
                if (run < 0) run = base;
                if (lane == (c0 >> 5)) bits |= ((1u << nch) - 1u) << (c0 & 31);
            }
            continue;
        }
#pragma unroll
        for (int u = 0; u < SX_BATCH; u++) {
            const int cb = base + 32 * u, i = cb + lane;
            if (cb >= nx) break;
            const bool set = i < nx && isfinite(v[u]);
            const unsigned ms = __ballot_sync(0xffffffffu, set);
            const int c = cb >> 5;
            if (!ms) {
                // no set cell in the chunk (most of a grid): filled at once when the walk is inside,
                // else part of the pending run and, so far, blank
                if (carry < 0) {
                    if (i < nx) d[i] = fillv;
                } else {
                    if (run < 0) run = cb;
                    if (lane == (c >> 5)) bits |= 1u << (c & 31);
                }
                continue;
            }
            const unsigned mn = __ballot_sync(0xffffffffu, set && v[u] < 0.0f);
            const int sl = state_from_left(ms, mn, lane, carry), sr = state_from_right(ms, mn, lane, 0);
            if (i < nx && !set && (sl < 0 || sr < 0)) d[i] = fillv;
            // the first set cell of the chunk decides the run pending from earlier chunks
            if (run >= 0 && ((mn >> (__ffs(ms) - 1)) & 1u)) {
                for (int x = run + lane; x < cb; x += 32) d[x] = fillv;
                bits &= ~chunk_mask(lane, run >> 5, c);                   // the pending chunks were filled after all
            }
            run = -1;
            carry = ((mn >> (31 - __clz(ms))) & 1u) ? -1 : 1;             // the last set cell of the chunk
            if (carry >= 0) {
                const int start = cb + 32 - __clz(ms);                    // first cell after the last set one
                if (start < min(nx, cb + 32)) run = start;
            }
        }
    }
    if (blank_y && lane < nwords) {
        const int64_t k = row / ny, j = row - k * ny;
        blank_y[(k * nwords + lane) * ny + j] = bits;        // along y for the y walk
        blank_z[(j * nwords + lane) * nz + k] = bits;        // along z for the z walk
    }
}

// ---- y and z: one thread per line, lines of a warp adjacent in x (coalesced); n cells, stride s.
// ONE walk does the work of the forward and the backward walk.  Within a sweep the two commute: a
// cell is filled iff the nearest set cell on either side is negative in the data at the start of the
// sweep (a forward fill never sits between an unset cell and its nearest set cell to the right
// unless that cell was filled by the same forward walk).  So the walk fills an unset cell at once
// when the last set cell was negative, and otherwise remembers where the unset run began and fills
// it when the next set cell turns out to be negative -- writes only, no second read of the line.
//
// The 32 lines of a warp share their 32-cell segment of every row, so the blank map says per (warp, row)
// whether the 32 cells are all unset: then they are not read (the walk of an unset cell needs no data).
// `mine` is the map laid out along this sweep's walk (word q of the line's run), fetched 32 rows at a
// time -- lane l takes row q0 + l, one ballot turns the 32 words into the skip mask of the warp.  A lane
// that fills a cell of a blank segment clears the bit in `next`, the map of the following sweep; that
// never happens on a well-resolved surface, where the x walk has already filled the whole interior.
#define SL_BATCH 8
__global__ void __launch_bounds__(256, 8) sweep_line_kernel(float *__restrict__ dist, int nx, int64_t outer_stride, int n,
                                                            int64_t stride, float fillv, int nwords,
                                                            const unsigned *__restrict__ mine,
                                                            unsigned *__restrict__ next, int64_t next_stride) {
    const int i = blockIdx.x * 256 + threadIdx.x, lane = threadIdx.x & 31;
    const int64_t o = blockIdx.y;
    const bool valid = i < nx;                  // lanes past the row end walk along, unset and silent
    float *d = dist + o * outer_stride + i;
    const int w = i >> 10;
    const unsigned bbit = 1u << ((i >> 5) & 31);
    if (mine) mine += (o * nwords + w) * (int64_t)n;
    if (next) next += (int64_t)w * (next_stride / nwords) + o;       // word of row (o, q): next[q * next_stride]
    int state = 0, run = -1;                 // run: first cell of the pending unset run, -1 = none
    unsigned ahead = (mine && lane < n) ? mine[lane] : 0u;
    for (int q32 = 0; q32 < n; q32 += 32) {
        const unsigned skipmask = __ballot_sync(0xffffffffu, (ahead & bbit) != 0u);
        ahead = (mine && q32 + 32 + lane < n) ? mine[q32 + 32 + lane] : 0u;
        const int qe = min(n, q32 + 32);
        if (skipmask == 0xffffffffu >> (32 - (qe - q32))) {
            // 32 blank rows: nothing to read, and (unless the walk is inside) nothing to write
            if (valid && state < 0) {
                for (int r = q32; r < qe; r++) {
                    d[(int64_t)r * stride] = fillv;
                    if (next) atomicAnd(&next[r * next_stride], ~bbit);
                }
            } else if (valid && run < 0) {
                run = q32;
            }
            continue;
        }
        for (int q0 = q32; q0 < qe; q0 += SL_BATCH) {
            float v[SL_BATCH];
#pragma unroll
            for (int u = 0; u < SL_BATCH; u++)
                v[u] = (valid && q0 + u < qe && !((skipmask >> (q0 + u - q32)) & 1u)) ? d[(int64_t)(q0 + u) * stride] : INFINITY;
#pragma unroll
            for (int u = 0; u < SL_BATCH; u++) {
                const int q = q0 + u;
                if (q >= qe) break;
                if (isfinite(v[u])) {
                    state = v[u] < 0.0f ? -1 : 1;
                    if (state < 0 && run >= 0)
                        for (int r = run; r < q; r++) {
                            d[(int64_t)r * stride] = fillv;
                            if (next && (next[r * next_stride] & bbit)) atomicAnd(&next[r * next_stride], ~bbit);
                        }
                    run = -1;
                } else if (!valid) {
                } else if (state < 0) {
                    d[(int64_t)q * stride] = fillv;
                    if (next && ((skipmask >> (q - q32)) & 1u)) atomicAnd(&next[q * next_stride], ~bbit);
                } else if (run < 0) {
                    run = q;
                }
            }
        }
    }
}

extern "C" int sdf_fill_interior(float *dist, int nx, int ny, int nz, float band, void *stream) {
    if (!dist || nx <= 0 || ny <= 0 || nz <= 0 || nx > 32767 || ny > 32767 || nz > 32767) return SDF_EINVAL;
    if (!(band > 0.0f) || !isfinite(band)) return SDF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { (void)cudaGetLastError(); return SDF_ECUDA; }
    cudaStream_t st = (cudaStream_t)stream;
    const float fillv = -band;
    const int64_t nrows = (int64_t)ny * nz;
    // blank maps: one bit per 32-cell segment, in y order and in z order (2/1024 of the grid),
    // stream-ordered scratch
    const int nwords = ((nx + 31) / 32 + 31) / 32;
    const size_t mapw = (size_t)nrows * nwords;
    unsigned *blank = nullptr;
    const char *pl = getenv("SDF_FILLINT_PLAIN");            // debug: every walk reads every cell
    if (!(pl && pl[0] == '1')) {
        // the maps come from the device's default memory pool; by default that pool hands everything back
        // to the driver at the next synchronisation and the allocation alone would cost more than the
        // sweeps: let it keep as much as the maps need (the one process-wide setting this call touches)
        const size_t need = sizeof(unsigned) * 2 * mapw;
        int dev = 0;
        cudaMemPool_t pool;
        CK(cudaGetDevice(&dev));
        CK(cudaDeviceGetDefaultMemPool(&pool, dev));
        unsigned long long keep = 0;
        CK(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
        if (keep < 2 * need + (64ull << 20)) {           // the pool reserves in chunks larger than the request
            keep = 2 * need + (64ull << 20);
            CK(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
        }
        CK(cudaMallocAsync((void **)&blank, need, st));
    }
    unsigned *by = blank, *bz = blank ? blank + mapw : nullptr;
    KL; sweep_x_kernel<<<(unsigned)((nrows + 7) / 8), 256, 0, st>>>(dist, nx, nrows, fillv, by, bz, nwords, ny, nz);
    // y: lines (i, k), cells nx apart;  z: lines (i, j), cells nx*ny apart.  A cell (j, k) filled by
    // the y walk clears word (j * nwords + w) * nz + k of the z map
    KL; sweep_line_kernel<<<dim3((unsigned)((nx + 255) / 256), (unsigned)nz), 256, 0, st>>>(
        dist, nx, (int64_t)nx * ny, ny, nx, fillv, nwords, by, bz, (int64_t)nwords * nz);
    KL; sweep_line_kernel<<<dim3((unsigned)((nx + 255) / 256), (unsigned)ny), 256, 0, st>>>(
        dist, nx, nx, nz, (int64_t)nx * ny, fillv, nwords, bz, nullptr, 0);
    cudaError_t e = cudaGetLastError();
    if (blank) cudaFreeAsync(blank, st);
    CK(e);
    return SDF_OK;
}

// ---------------------------------------------------------------------------------------
// sdf_fill_interior_static: the same three sweeps for callers that must not allocate (CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc).  The blank maps live in a file-scope device array instead of the
// stream-ordered pool: SDF_FILL_STATIC_BYTES per GPU that loads the library, held until the process exits.
//   - grids whose maps do not fit (more than ny * nz * ceil(nx / 1024) = 2^20 map words) are refused: SDF_ETOOBIG
//   - no cudaMalloc / cudaFree / cudaMallocAsync / pool call on any path of this function
//   - every call uses the SAME array: calls that overlap on the GPU (different streams without an order between
//     them, or different host threads) race on it.  The array keeps the last call's contents; nothing has to be cleared:
//     sweep_x_kernel writes every map word of this call's grid before the y and z walks read one.
// In host code `g_fill_static_maps` is only the symbol's host-side stand-in: its device address is looked up once per
// device (with that device current) through cudaGetSymbolAddress and that pointer is what the kernels get.
// ---------------------------------------------------------------------------------------
#define SDF_FILL_STATIC_BYTES (8u << 20)      /* 1024^3 cells (C4): 2 maps x 2^20 words x 4 B */
static __device__ __align__(256) unsigned g_fill_static_maps[SDF_FILL_STATIC_BYTES / sizeof(unsigned)];

#define FILL_STATIC_MAX_DEVICES 64
static unsigned *g_fill_static_ptr[FILL_STATIC_MAX_DEVICES];      // per device: address of the array (0 = not looked up yet)

extern "C" int sdf_fill_interior_static(float *dist, int nx, int ny, int nz, float band, void *stream) {
    if (!dist || nx <= 0 || ny <= 0 || nz <= 0 || nx > 32767 || ny > 32767 || nz > 32767) return SDF_EINVAL;
    if (!(band > 0.0f) || !isfinite(band)) return SDF_EINVAL;
    const int64_t nrows = (int64_t)ny * nz;
    const int nwords = ((nx + 31) / 32 + 31) / 32;
    const size_t mapw = (size_t)nrows * nwords;
    if (sizeof(unsigned) * 2 * mapw > (size_t)SDF_FILL_STATIC_BYTES) return SDF_ETOOBIG;
    int ndev = 0, dev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { (void)cudaGetLastError(); return SDF_ECUDA; }
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= FILL_STATIC_MAX_DEVICES) return SDF_EINVAL;
    unsigned *maps = g_fill_static_ptr[dev];
    if (!maps) {
        // set-up, once per device (two host threads arriving together look the same address up twice)
        CK(cudaGetSymbolAddress((void **)&maps, g_fill_static_maps));
        if (!maps) return SDF_ECUDA;
        g_fill_static_ptr[dev] = maps;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const float fillv = -band;
    unsigned *by = maps, *bz = maps + mapw;
    KL; sweep_x_kernel<<<(unsigned)((nrows + 7) / 8), 256, 0, st>>>(dist, nx, nrows, fillv, by, bz, nwords, ny, nz);
    KL; sweep_line_kernel<<<dim3((unsigned)((nx + 255) / 256), (unsigned)nz), 256, 0, st>>>(
        dist, nx, (int64_t)nx * ny, ny, nx, fillv, nwords, by, bz, (int64_t)nwords * nz);
    KL; sweep_line_kernel<<<dim3((unsigned)((nx + 255) / 256), (unsigned)ny), 256, 0, st>>>(
        dist, nx, nx, nz, (int64_t)nx * ny, fillv, nwords, bz, nullptr, 0);
    CK(cudaGetLastError());
    return SDF_OK;
}
