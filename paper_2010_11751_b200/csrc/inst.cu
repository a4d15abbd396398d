// inst.cu -- step kernels of ONE (lattice, collision model) pair; compiled once per pair with
//   -DLBM_INST_Q=<19|27> -DLBM_INST_MODEL=<0..9>
// (see paper_2010_11751_b200/build.py).  fp64 always; fp32 for the W2 family (BGK_W2, TRT, REG).
#include "dispatch.cuh"

#ifndef LBM_INST_Q
#error "compile with -DLBM_INST_Q=19|27 -DLBM_INST_MODEL=0..9"
#endif

namespace lbm {

template <class T, int Q, int MODEL, bool SOA>
static cudaError_t launch_kind(int kind, int block, const StepArgs<T>& a, cudaStream_t s)
{
    const int grid = (a.g.n + block - 1) / block;
    switch (kind) {
    case SK_PUSH: step_kernel<T, Q, MODEL, SOA, LD_LOCAL, ST_PUSH><<<grid, block, 0, s>>>(a); break;
    case SK_PULL: step_kernel<T, Q, MODEL, SOA, LD_PULL, ST_LOCAL><<<grid, block, 0, s>>>(a); break;
    case SK_COLLIDE: step_kernel<T, Q, MODEL, SOA, LD_LOCAL, ST_LOCAL><<<grid, block, 0, s>>>(a); break;
    case SK_EVEN: step_kernel<T, Q, MODEL, SOA, LD_LOCAL, ST_SWAPPED><<<grid, block, 0, s>>>(a); break;
    case SK_ODD: step_kernel<T, Q, MODEL, SOA, LD_AAPULL, ST_PUSH><<<grid, block, 0, s>>>(a); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

template <class T, int Q, int MODEL>
cudaError_t launch_step(int kind, bool soa, int block, const StepArgs<T>& a, cudaStream_t s)
{
    if (block <= 0 || block > 256 || (block & 31)) return cudaErrorInvalidValue;
    return soa ? launch_kind<T, Q, MODEL, true>(kind, block, a, s) : launch_kind<T, Q, MODEL, false>(kind, block, a, s);
}

template cudaError_t launch_step<double, LBM_INST_Q, LBM_INST_MODEL>(int, bool, int, const StepArgs<double>&, cudaStream_t);
#if LBM_INST_MODEL == 0 || LBM_INST_MODEL == 2 || LBM_INST_MODEL == 9
template cudaError_t launch_step<float, LBM_INST_Q, LBM_INST_MODEL>(int, bool, int, const StepArgs<float>&, cudaStream_t);
#endif

}  // namespace lbm
