// inst.cu -- step kernels of ONE (lattice, collision model) pair; compiled once per pair with
//   -DLBM_INST_Q=<19|27> -DLBM_INST_MODEL=<0..14>  (collision.cuh: enum Model)
// (see paper_2010_11751_b200/build.py).  fp64 and fp32 (shifted storage, R20).
#include "dispatch.cuh"
#include "tma_step.cuh"
#include "aos_march.cuh"

#ifndef LBM_INST_Q
#error "compile with -DLBM_INST_Q=19|27 -DLBM_INST_MODEL=0..14"
#endif

namespace lbm {

template <class T, int Q, int MODEL, bool SOA, int LOAD, int STORE>
static cudaError_t launch_one(int block, bool staged, const StepArgs<T>& a, cudaStream_t s)
{
    // AoS two-population pull, whole lattice, outermost x-layers solid: neighbour records staged in a
    // marching shared-memory tile (aos_march.cuh)
    if constexpr (!SOA && LOAD == LD_PULL && STORE == ST_LOCAL) {
        if (a.march && staged && a.first == 0 && a.end == a.g.n && a.g.nx >= 4) {
            constexpr int TY = 4, TZ = 32;
            using G = MarchGeo<T, Q, TY, TZ>;
            auto kernel = step_kernel_aos_march<T, Q, MODEL, TY, TZ>;
            static int per_sm = 0, sms = 0;   // per instantiation
            if (!per_sm) {
                cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM);
                if (e != cudaSuccess) return e;
                int dev = 0;
                cudaGetDevice(&dev);
                cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
                e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, TY * TZ, G::SMEM);
                if (e != cudaSuccess || per_sm < 1) { per_sm = 0; return e != cudaSuccess ? e : cudaErrorLaunchOutOfResources; }
            }
            const int tz = (a.g.nz + TZ - 1) / TZ, ty = (a.g.ny + TY - 1) / TY;
            // x-segments: enough blocks for a few waves; a segment re-reads two layers, so keep it long
            int nseg = (4 * per_sm * sms + tz * ty - 1) / (tz * ty);
            const int max_seg = (a.g.nx - 2 + 15) / 16;
            if (nseg > max_seg) nseg = max_seg;
            if (nseg < 1) nseg = 1;
            const int xlen = (a.g.nx - 2 + nseg - 1) / nseg;
            nseg = (a.g.nx - 2 + xlen - 1) / xlen;
            kernel<<<dim3(tz, ty, nseg), TY * TZ, G::SMEM, s>>>(a, xlen);
            return cudaGetLastError();
        }
    }
    // AoS two-population pull, whole lattice: blocks cover patches of z-rows so that source rows are shared in L1
    if constexpr (!SOA && LOAD == LD_PULL && STORE == ST_LOCAL) {
        if (a.patch && staged && a.first == 0 && a.end == a.g.n) {
            constexpr int PY = LBM_AOS_PATCH_PY;
            const dim3 grid = patch_grid(a.g, PY);
            const size_t smem = ((size_t)32 * PY * Q + (size_t)96 * PY) * sizeof(T);
            auto kernel = step_kernel_aos_pull_patch<T, Q, MODEL, PY>;
            if (smem > 48 * 1024) {
                static bool raised = false;   // per instantiation
                if (!raised) {
                    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
                    if (e != cudaSuccess) return e;
                    raised = true;
                }
            }
            kernel<<<grid, 32 * PY, smem, s>>>(a);
            return cudaGetLastError();
        }
    }
    // AoS AA odd step, whole lattice: cooperative gather and scatter of the z-triples (kernels.cuh)
    if constexpr (!SOA && LOAD == LD_AAPULL && STORE == ST_PUSH) {
        if (staged && a.first == 0 && a.end == a.g.n) {
            static_assert(LBM_AOS_PATCH_PY == 4, "step_kernel_aos_odd has 128 threads");
            if (a.patch) {
                step_kernel_aos_odd<T, Q, MODEL, true><<<patch_grid(a.g, LBM_AOS_PATCH_PY), 128, (size_t)4 * 96 * sizeof(T), s>>>(a);
                return cudaGetLastError();
            }
            const int b = block > 128 ? 128 : block;
            step_kernel_aos_odd<T, Q, MODEL><<<(a.g.n + b - 1) / b, b, (size_t)(b / 32) * 96 * sizeof(T), s>>>(a);
            return cudaGetLastError();
        }
    }
    if constexpr (!SOA && (LOAD == LD_LOCAL || STORE != ST_PUSH)) {
        if (staged && a.first == 0 && a.end == a.g.n) {  // AoS: local accesses through a transposing shared-memory tile (kernels.cuh)
            const int b = block > 128 ? 128 : block;
            step_kernel_aos<T, Q, MODEL, LOAD, STORE><<<(a.g.n + b - 1) / b, b, ((size_t)b * Q + (size_t)(b / 32) * 96) * sizeof(T), s>>>(a);
            return cudaGetLastError();
        }
    }
    // SoA, whole lattice: loads staged through shared memory by the TMA unit (tma_step.cuh)
    if constexpr (SOA && ((LOAD == LD_PULL && STORE == ST_LOCAL) || (LOAD == LD_LOCAL && STORE == ST_SWAPPED) ||
                          (LOAD == LD_AAPULL && STORE == ST_PUSH))) {
        if (a.tma && a.first == 0 && a.end == a.g.n) {
            constexpr int B = tma_tile<T, Q>(), S = tma_stages<T, Q>();
            constexpr size_t smem = tma_smem_bytes<T, Q, B, S>();
            auto kernel = step_kernel_tma<T, Q, MODEL, LOAD, STORE>;
            static int per_sm = 0, sms = 0;   // per instantiation
            if (!per_sm) {
                cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
                if (e != cudaSuccess) return e;
                int dev = 0;
                cudaGetDevice(&dev);
                cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
                e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, B, smem);
                if (e != cudaSuccess || per_sm < 1) { per_sm = 0; return e != cudaSuccess ? e : cudaErrorLaunchOutOfResources; }
            }
            const int ntiles = (a.g.n + B - 1) / B;
            const int grid = ntiles < per_sm * sms ? ntiles : per_sm * sms;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)grid);
            cfg.blockDim = dim3((unsigned)B);
            cfg.dynamicSmemBytes = smem;
            cfg.stream = s;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = attr;
            cfg.numAttrs = a.pdl ? 1 : 0;
            return cudaLaunchKernelEx(&cfg, kernel, a);
        }
    }
    const int b = block > max_threads<T, Q>() ? max_threads<T, Q>() : block;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((a.end - a.first + b - 1) / b));
    cfg.blockDim = dim3((unsigned)b);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = a.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, step_kernel<T, Q, MODEL, SOA, LOAD, STORE>, a);
}

template <class T, int Q, int MODEL, bool SOA>
static cudaError_t launch_kind(int kind, int block, bool staged, const StepArgs<T>& a, cudaStream_t s)
{
    switch (kind) {
    case SK_PUSH: return launch_one<T, Q, MODEL, SOA, LD_LOCAL, ST_PUSH>(block, staged, a, s);
    case SK_PULL: return launch_one<T, Q, MODEL, SOA, LD_PULL, ST_LOCAL>(block, staged, a, s);
    case SK_COLLIDE: return launch_one<T, Q, MODEL, SOA, LD_LOCAL, ST_LOCAL>(block, staged, a, s);
    case SK_EVEN: return launch_one<T, Q, MODEL, SOA, LD_LOCAL, ST_SWAPPED>(block, staged, a, s);
    case SK_ODD: return launch_one<T, Q, MODEL, SOA, LD_AAPULL, ST_PUSH>(block, staged, a, s);
    default: return cudaErrorInvalidValue;
    }
}

template <class T, int Q, int MODEL>
cudaError_t launch_step(int kind, bool soa, int block, bool staged, const StepArgs<T>& a, cudaStream_t s)
{
    if (block <= 0 || block > 256 || (block & 31)) return cudaErrorInvalidValue;
    return soa ? launch_kind<T, Q, MODEL, true>(kind, block, staged, a, s) : launch_kind<T, Q, MODEL, false>(kind, block, staged, a, s);
}

template cudaError_t launch_step<double, LBM_INST_Q, LBM_INST_MODEL>(int, bool, int, bool, const StepArgs<double>&, cudaStream_t);
template cudaError_t launch_step<float, LBM_INST_Q, LBM_INST_MODEL>(int, bool, int, bool, const StepArgs<float>&, cudaStream_t);

}  // namespace lbm
