// cdp.cu -- ABLATION, off by default: the paper's dynamic-parallelism
// scheduler (sec.9.1, Table 3): "a single kernel from the host, assigning a single
// thread for each bounding volume which dynamically launch kernels with a thread per cell".
//
//   SDF_SCHEDULER=dynamic      every live polyhedron launches a child grid, one thread per cell of
//                              its bounding volume (the configuration of Table 3)
//   SDF_SCHEDULER=dynamic:N    hybrid (the "optimal implementation" of PAPER.md:470, after Tang et
//                              al.): bounding volumes of at most N cells are walked serially by the
//                              parent thread, larger ones get a child grid
//
// The only translation unit built as relocatable device code (device-side launches need the
// device runtime); it shares the arithmetic of evaluate.cuh with the default kernels, so the
// candidates and the packed atomicMin are the same and only the schedule differs.  The parent is
// launched in chunks so that the children of one chunk fit the device runtime's pending-launch
// pool; a child launch the runtime refuses is counted (CTR_CDP_FALLBACK) and its volume is walked
// by the parent thread, so the result never depends on the pool.  DESIGN.md sec.12 has the numbers.
#include "evaluate.cuh"

struct CdpParams {
    MeshView mv;
    GridParams g;
    const int *table;
    u64 *scratch;
    u64 *ctr;
};

#define CDP_BT 128
#define CDP_CHUNK 65536          // polyhedra per parent launch

// child: one thread per cell of the bounding volume ("threads are launched according
// to the size of the volume and the domain coordinates of each thread can be determined from the
// limits of the bounding volume"); the cell is a bounding volume of one cell for the serial walk
__global__ void __launch_bounds__(CDP_BT) cdp_child_kernel(const CdpParams *__restrict__ P, int64_t p, PolyHdr H) {
    const int ni = H.i1 - H.i0 + 1, nj = H.j1 - H.j0 + 1, nk = H.k1 - H.k0 + 1;
    const int64_t c = (int64_t)blockIdx.x * CDP_BT + threadIdx.x;
    if (c >= (int64_t)ni * nj * nk) return;
    PolyHdr one;
    one.i0 = one.i1 = (short)(H.i0 + (int)(c % ni));
    one.j0 = one.j1 = (short)(H.j0 + (int)((c / ni) % nj));
    one.k0 = one.k1 = (short)(H.k0 + (int)(c / ((int64_t)ni * nj)));
    one.rows = 1;
    one.msin = H.msin;
    u32 tested = 0, accepted = 0;
    process_direct(P->mv, P->g, p, one, P->table, P->scratch, tested, accepted);
}

// parent: one thread per polyhedron
__global__ void __launch_bounds__(CDP_BT) cdp_parent_kernel(const CdpParams *__restrict__ P, int64_t first, int64_t count,
                                                            int64_t serial_below) {
    const int64_t q = (int64_t)blockIdx.x * CDP_BT + threadIdx.x;
    if (q >= count) return;
    const int64_t p = first + q;
    PolyHdr H;
    if (!poly_aabv(P->mv, P->g, p, H)) return;
    const int64_t cells = (int64_t)(H.i1 - H.i0 + 1) * (int64_t)H.rows;
    bool serial = cells <= serial_below;
    if (!serial) {
        cdp_child_kernel<<<(unsigned)((cells + CDP_BT - 1) / CDP_BT), CDP_BT, 0, cudaStreamFireAndForget>>>(P, p, H);
        if (cudaGetLastError() != cudaSuccess) {          // pending-launch pool exhausted
            atomicAdd(&P->ctr[CTR_CDP_FALLBACK], 1ull);
            serial = true;
        }
    }
    if (serial) {
        u32 tested = 0, accepted = 0;
        process_direct(P->mv, P->g, p, H, P->table, P->scratch, tested, accepted);
    }
}

int run_cdp_evaluate(sdf_mesh *m, const MeshView &mv, const GridParams &g, cudaStream_t st) {
    static int pool_set = 0;
    if (!pool_set) {
        CK(cudaDeviceSetLimit(cudaLimitDevRuntimePendingLaunchCount, CDP_CHUNK + 4096));
        pool_set = 1;
    }
    CdpParams hp;
    hp.mv = mv; hp.g = g; hp.table = m->brick_table; hp.scratch = m->scratch; hp.ctr = m->d_ctr;
    CdpParams *dp = nullptr;
    CKS(dev_alloc(&m->alloc, (void **)&dp, sizeof(CdpParams), st));
    cudaError_t e = cudaMemcpyAsync(dp, &hp, sizeof(hp), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);          // hp lives on this stack frame
    for (int64_t first = 0; e == cudaSuccess && first < mv.P; first += CDP_CHUNK) {
        const int64_t count = mv.P - first < CDP_CHUNK ? mv.P - first : CDP_CHUNK;
        KL; cdp_parent_kernel<<<(unsigned)((count + CDP_BT - 1) / CDP_BT), CDP_BT, 0, st>>>(dp, first, count, (int64_t)g.cdp_serial_below);
        e = cudaGetLastError();
    }
    dev_free(&m->alloc, dp, st);
    if (e != cudaSuccess) { CK(e); }
    return SDF_OK;
}
