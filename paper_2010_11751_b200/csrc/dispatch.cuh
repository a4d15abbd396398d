// dispatch.cuh -- host-side launch entry points shared by lbm_api.cu (caller), inst.cu (one object
// per lattice x collision model: the step kernels) and aux.cu (model-independent kernels).
#pragma once
#include <cuda_runtime.h>
#include "kernels.cuh"

namespace lbm {

// step-kernel kinds = (load mode, store mode) pairs, see kernels.cuh
enum StepKind {
    SK_PUSH = 0,   // LD_LOCAL  -> ST_PUSH     two-population, collide then push (Table 1)
    SK_PULL,       // LD_PULL   -> ST_LOCAL    two-population, pull then collide (post-collision storage)
    SK_COLLIDE,    // LD_LOCAL  -> ST_LOCAL    collide only (first step of the pull form)
    SK_EVEN,       // LD_LOCAL  -> ST_SWAPPED  AA even step / swap pass 1 (Table 1)
    SK_ODD,        // LD_AAPULL -> ST_PUSH     AA odd step (Table 1)
    SK_COUNT
};

// implementation variants of the step kernels (lbm_set_variant)
enum Variant {
    V_DEFAULT = 0,   // library's choice
    V_GENERIC_PUSH,  // generic one-thread-per-cell kernels, 2-pop as collide-then-push
    V_GENERIC_PULL,  // generic kernels, 2-pop as pull-then-collide with lazily streamed storage
    V_AOS_PLAIN,     // AoS without the shared-memory tile (every access a per-thread gather / scatter)
    V_TMA,           // SoA: loads staged through shared memory by TMA bulk copies (tma_step.cuh)
    V_NO_TMA,        // SoA: never that kernel (one cell per thread, loads into registers, L2 prefetch)
    V_PLAIN,         // as V_NO_TMA, and neither L2 prefetch nor programmatic dependent launch nor the alternating traversal
                     // direction (pure scheduling: same results)
    V_AOS_MARCH,     // AoS two-population pull: neighbour records in a marching shared-memory tile (aos_march.cuh)
    V_COUNT
};

// defined in inst.cu, explicitly instantiated once per (T, Q, MODEL)
template <class T, int Q, int MODEL>
cudaError_t launch_step(int kind, bool soa, int block, bool staged, const StepArgs<T>& a, cudaStream_t s);

// defined in aux.cu
// flags -> code bytes + per-group edge bits and ordinals (+ the number of edge cells in total[0]); then the
// compact mask array, which the caller allocates from that number
cudaError_t aux_classify_codes(int Q, const uint8_t* flags, uint8_t* code, uint2* grp, unsigned* total, unsigned* sums,
                               const Geo& g, cudaStream_t s);
cudaError_t aux_classify_masks(int Q, const uint8_t* flags, const uint8_t* code, const uint2* grp, unsigned long long* mask,
                               const Geo& g, cudaStream_t s);
template <class T>
cudaError_t aux_init_equilibrium(int Q, bool ext, bool soa, T* pop, const uint8_t* code, const Geo& g, const T* rho,
                                 const T* u, cudaStream_t s);
template <class T>
cudaError_t aux_macroscopic(int Q, bool soa, int load, const StepArgs<T>& a, T* rho, T* u, cudaStream_t s);
enum { ENERGY_STAGE2 = 512 };  // blocks of the second reduction stage
template <class T>
cudaError_t aux_energy(int Q, bool soa, int load, const StepArgs<T>& a, double* partial, int nblocks, double* out,
                       cudaStream_t s);
template <class T>
cudaError_t aux_extract_plane(int Q, bool soa, const T* pop, const uint8_t* code, const Geo& g, const PlaneArgs& p,
                              T* out, const int* cells, int m, cudaStream_t s);
template <class T>
cudaError_t aux_insert_plane(int Q, bool soa, T* pop, const uint8_t* code, const Geo& g, int k, double weight,
                             const T* in, cudaStream_t s);
template <class T>
cudaError_t aux_swap_stream(int Q, bool soa, const StepArgs<T>& a, cudaStream_t s);
template <class T>
cudaError_t aux_halo(bool pack, T* pop, const uint8_t* code, long long stride, const HaloArgs& p, T* buf, cudaStream_t s);
// stream only (LD_PULL -> ST_LOCAL without collision): turns post-collision storage into canonical
template <class T>
cudaError_t aux_stream_only(int Q, bool soa, const StepArgs<T>& a, cudaStream_t s);

// host copies of the lattice tables (from Lat<Q>); aos[k] = slot of direction k inside an AoS record
void lattice_tables(int Q, int (*c)[3], int* opp, double* w, int* aos);

}  // namespace lbm
