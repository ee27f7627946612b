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

#define SX_BATCH 8       // chunks of 32 cells loaded before they are resolved (memory-level parallelism)
// One walk per row (see sweep_line_kernel for why one is enough).  A chunk of 32 cells is resolved
// with two ballots: an unset cell is filled if the nearest set cell to its left (in the chunk, else
// the carry) or to its right IN THE CHUNK is negative; unset cells with no set cell to their right
// in the chunk join the pending run, which the first set cell of a later chunk resolves (the warp
// then fills the earlier chunks' part of the run with coalesced stores).
__global__ void __launch_bounds__(256) sweep_x_kernel(float *__restrict__ dist, int nx, int64_t nrows, float fillv) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (row >= nrows) return;
    float *d = dist + row * nx;
    int carry = 0, run = -1;
    for (int base = 0; base < nx; base += 32 * SX_BATCH) {
        float v[SX_BATCH];
#pragma unroll
        for (int u = 0; u < SX_BATCH; u++) {
            const int i = base + 32 * u + lane;
            v[u] = i < nx ? d[i] : INFINITY;
        }
#pragma unroll
        for (int u = 0; u < SX_BATCH; u++) {
            const int cb = base + 32 * u, i = cb + lane;
            if (cb >= nx) break;
            const bool set = i < nx && isfinite(v[u]);
            const unsigned ms = __ballot_sync(0xffffffffu, set), mn = __ballot_sync(0xffffffffu, set && v[u] < 0.0f);
            const int sl = state_from_left(ms, mn, lane, carry), sr = state_from_right(ms, mn, lane, 0);
            if (i < nx && !set && (sl < 0 || sr < 0)) d[i] = fillv;
            if (ms) {
                // the first set cell of the chunk decides the run pending from earlier chunks
                if (run >= 0 && ((mn >> (__ffs(ms) - 1)) & 1u))
                    for (int x = run + lane; x < cb; x += 32) d[x] = fillv;
                run = -1;
            }
            carry = state_from_left(ms, mn, 31, carry);
            if (carry >= 0 && run < 0) {
                const int start = cb + (ms ? 32 - __clz(ms) : 0);       // first cell after the last set one
                if (start < min(nx, cb + 32)) run = start;
            }
        }
    }
}

// ---- y and z: one thread per line, lines of a warp adjacent in x (coalesced); n cells, stride s.
// ONE walk does the work of the forward and the backward walk.  Within a sweep the two commute: a
// cell is filled iff the nearest set cell on either side is negative in the data at the start of the
// sweep (a forward fill never sits between an unset cell and its nearest set cell to the right
// unless that cell was filled by the same forward walk).  So the walk fills an unset cell at once
// when the last set cell was negative, and otherwise remembers where the unset run began and fills
// it when the next set cell turns out to be negative -- writes only, no second read of the line.
#define SL_BATCH 8
__global__ void __launch_bounds__(256) sweep_line_kernel(float *__restrict__ dist, int nx, int64_t nlines_outer,
                                                         int64_t outer_stride, int n, int64_t stride, float fillv) {
    const int i = blockIdx.x * 256 + threadIdx.x;
    const int64_t o = blockIdx.y;
    if (i >= nx || o >= nlines_outer) return;
    float *d = dist + o * outer_stride + i;
    int state = 0, run = -1;                 // run: first cell of the pending unset run, -1 = none
    for (int q0 = 0; q0 < n; q0 += SL_BATCH) {
        float v[SL_BATCH];
#pragma unroll
        for (int u = 0; u < SL_BATCH; u++) v[u] = (q0 + u < n) ? d[(int64_t)(q0 + u) * stride] : INFINITY;
#pragma unroll
        for (int u = 0; u < SL_BATCH; u++) {
            const int q = q0 + u;
            if (q >= n) break;
            if (isfinite(v[u])) {
                state = v[u] < 0.0f ? -1 : 1;
                if (state < 0 && run >= 0)
                    for (int r = run; r < q; r++) d[(int64_t)r * stride] = fillv;
                run = -1;
            } else if (state < 0) {
                d[(int64_t)q * stride] = fillv;
            } else if (run < 0) {
                run = q;
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
    KL; sweep_x_kernel<<<(unsigned)((nrows + 7) / 8), 256, 0, st>>>(dist, nx, nrows, fillv);
    // y: lines (i, k), cells nx apart;  z: lines (i, j), cells nx*ny apart
    KL; sweep_line_kernel<<<dim3((unsigned)((nx + 255) / 256), (unsigned)nz), 256, 0, st>>>(
        dist, nx, nz, (int64_t)nx * ny, ny, nx, fillv);
    KL; sweep_line_kernel<<<dim3((unsigned)((nx + 255) / 256), (unsigned)ny), 256, 0, st>>>(
        dist, nx, ny, nx, nz, (int64_t)nx * ny, fillv);
    CK(cudaGetLastError());
    return SDF_OK;
}
