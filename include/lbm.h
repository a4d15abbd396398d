/*
 * lbm.h -- C ABI of the B200-native lattice Boltzmann stream-and-collide library
 * (liblbm_b200.so), after arxiv 2010.11751 (Latt, Coreixas, Beny).  Citations "PAPER.md:Lnnn"
 * are lines of the paper text; "R<n>" are the readings listed in DESIGN.md.
 *
 * Conventions shared by every call
 *   - Host arrays are indexed i = (ix*ny + iy)*nz + iz, z fastest.
 *     u is three planes [3][N]; populations are [Q][N] in the canonical direction order (R7):
 *     D3Q19: k=0..8 = (-1,0,0),(0,-1,0),(0,0,-1),(-1,-1,0),(-1,1,0),(-1,0,-1),(-1,0,1),(0,-1,-1),
 *     (0,-1,1); k=9 rest; k=10..18 their negatives.  D3Q27 appends (-1,-1,-1),(-1,-1,1),(-1,1,-1),
 *     (-1,1,1) to the half set (rest at 13, opposite of k is k+14).  The internal device layout
 *     (padding, AoS, AA shuffling, post-collision storage) is never visible.
 *   - "host" pointers are caller-owned and only read / written during the call.  The context owns
 *     every device buffer; device memory and the stream come from the hooks (lbm_set_hooks), which
 *     the Python binding points at torch's caching allocator and current stream.
 *   - Index arithmetic wraps periodically on all three axes; walls exist only where flags say so
 *     (a cavity is a box whose outermost layer is flagged).
 *   - Non-fluid cells export populations 0, rho 0, u 0.
 *   - Return value: 0 ok; LBM_E_ARG (-1) bad argument / unsupported combination; LBM_E_ALLOC (-2);
 *     LBM_E_CUDA (-3); LBM_E_STATE (-4) wrong state (e.g. step before init).  lbm_create returns
 *     NULL on failure.  The message is available from lbm_last_error() (thread-local).  Nothing
 *     throws or aborts across this boundary, and there is no CPU fallback of any kind.
 *   - One context = one stream; calls on one context are not re-entrant.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbm_ctx lbm_t;

enum { LBM_D3Q19 = 19, LBM_D3Q27 = 27 };
/* collision models: the paper's nine plus regularised BGK (R18) */
enum { LBM_BGK_W2 = 0, LBM_BGK_NW4, LBM_TRT, LBM_RM, LBM_HM, LBM_CM, LBM_CHM, LBM_K, LBM_RR, LBM_REG, LBM_NUM_MODELS };
/* memory-access schemes x layouts (Table 1) */
enum { LBM_2POP_SOA = 0, LBM_2POP_AOS, LBM_SWAP_SOA, LBM_SWAP_AOS, LBM_AA_SOA, LBM_AA_AOS, LBM_NUM_SCHEMES };
enum { LBM_F32 = 0, LBM_F64 = 1 };
enum { LBM_FLUID = 0, LBM_WALL = 1, LBM_MOVING = 2, LBM_GHOST = 3 }; /* cell flags; LBM_GHOST = a
   fluid cell owned by another rank of a slab decomposition: never updated and left out of every
   sum and export, read like a fluid cell by its neighbours, filled by lbm_halo_unpack */
enum { LBM_OK = 0, LBM_E_ARG = -1, LBM_E_ALLOC = -2, LBM_E_CUDA = -3, LBM_E_STATE = -4 };

/* Device-memory and stream hooks (process-wide; set before lbm_create).  alloc returns a device
 * pointer of at least `bytes` bytes aligned to 256 B or NULL; free releases it; stream is a
 * cudaStream_t (as void*) on which every kernel and copy of contexts created afterwards runs.
 * With no hooks set the library uses cudaMalloc/cudaFree and the legacy default stream. */
typedef void* (*lbm_alloc_fn)(size_t bytes);
typedef void (*lbm_free_fn)(void* ptr);
int lbm_set_hooks(lbm_alloc_fn alloc, lbm_free_fn free_fn, void* stream);

/* Create a context for an nx*ny*nz box (each >= 3), lattice LBM_D3Q19|LBM_D3Q27, a collision
 * model, a scheme, the shear relaxation rate omega in (0,2) with nu = (1/omega - 1/2)/3
 * and the storage/arithmetic type.  All cells start FLUID (fully periodic box).
 * Default rates (R14): omega_bulk = omega, moments of order >= 3 relaxed with 1 (RR: with omega);
 * TRT magic parameter 1/4 (R15).  LBM_F32 stores and computes on f_k - t_k (R20). */
lbm_t* lbm_create(int nx, int ny, int nz, int lattice, int collision, int scheme, double omega, int dtype);
int lbm_destroy(lbm_t* ctx);

/* Cell flags (host, uint8 [N]) and the velocity of LBM_MOVING cells (host double[3], may be NULL
 * = 0).  Half-way bounce-back with the momentum term -6 t_k rho_w c_k.u_w, rho_w = 1, Eq 3
 * (PAPER.md:L87-92).  Must precede lbm_init_equilibrium / lbm_set_populations. */
int lbm_set_flags(lbm_t* ctx, const uint8_t* flags, const double u_wall[3]);

/* Override the rates of Eq 11 / Eq 13-15: bulk rate, rate of third-order
 * moments, rate of moments of order >= 4.  Ignored by BGK_W2, BGK_NW4, TRT and REG. */
int lbm_set_relaxation(lbm_t* ctx, double omega_bulk, double omega3, double omega_hi);
/* TRT magic parameter Lambda = (1/w+ - 1/2)(1/w- - 1/2) (default 1/4). */
int lbm_set_trt_magic(lbm_t* ctx, double lambda);

/* Fill every fluid cell with the model's own equilibrium (Eq 6 for BGK_W2/TRT/REG, the extended
 * product-form equilibrium for the rest) of the given rho [N] and u [3][N]: host arrays of the
 * context dtype.  Resets the step count and the AA parity. */
int lbm_init_equilibrium(lbm_t* ctx, const void* rho, const void* u);

/* Same with rho [N] and u [3][N] already in DEVICE memory (context dtype, 16 B aligned);
 * asynchronous on the stream; the buffers must stay valid until the stream reaches this point. */
int lbm_init_equilibrium_device(lbm_t* ctx, const void* rho_dev, const void* u_dev);

/* n collide-and-stream cycles (Eq 1-3) by the context's scheme; asynchronous on
 * the stream.  n >= 0. */
int lbm_step(lbm_t* ctx, int n);

/* rho = sum_k f_k, u = sum_k c_k f_k / rho per cell of the pre-collision
 * populations at the current time; host outputs of the context dtype; synchronises. */
int lbm_macroscopic(lbm_t* ctx, void* rho, void* u);

/* Same into DEVICE buffers rho_dev [N], u_dev [3][N]; asynchronous on the stream. */
int lbm_macroscopic_device(lbm_t* ctx, void* rho_dev, void* u_dev);

/* E = sum over fluid cells of 1/2 rho |u|^2 (R19), accumulated in double with a fixed reduction
 * tree (bitwise repeatable); synchronises. */
int lbm_kinetic_energy(lbm_t* ctx, double* e);
/* Same into one double in DEVICE memory; asynchronous on the stream. */
int lbm_kinetic_energy_device(lbm_t* ctx, double* e_dev);

/* The same reduction through an entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc
 * (code under CUDA-graph capture, tight serving loops, harnesses that forbid it): the per-block partial
 * sums live in a fixed array of LBM_STATIC_SCRATCH_DOUBLES doubles (2 MiB) in the library's device image,
 * which every GPU that loads the library holds until the process exits.  Same kernels and the same fixed
 * reduction tree as lbm_kinetic_energy_device, so the result is bit for bit the same; e_dev = one double in
 * DEVICE memory; asynchronous on the stream; calls no cudaMalloc / cudaFree / allocating library routine
 * (the first call on a device resolves the array's address with cudaGetSymbolAddress).
 * Limit: lattices of at most LBM_STATIC_MAX_CELLS cells (66 977 792, e.g. 406^3); larger ones return LBM_E_ARG
 * with a message naming the limit.  The array is shared by every context and every call on a device and
 * keeps the last call's contents (nothing in it needs clearing: a call reads only what it has written);
 * calls that overlap on the GPU -- two contexts on different streams of one device -- RACE on it: order
 * them on one stream or with events. */
#define LBM_STATIC_SCRATCH_DOUBLES 262144
#define LBM_STATIC_MAX_CELLS ((LBM_STATIC_SCRATCH_DOUBLES - 512LL) * 256LL)
int lbm_kinetic_energy_device_static(lbm_t* ctx, double* e_dev);

/* Pre-collision populations at the current time, canonical [Q][N] order, context dtype, host. */
int lbm_get_populations(lbm_t* ctx, void* f);
/* The same for m listed cells only: cells = host int32 [m] of cell indices in [0, N), f = host
 * [Q][m] of the context dtype (f[k*m + t] = f_k(cells[t])).  Lets the parity tests sample a
 * 512^3 lattice without a 20 GB export.  0 <= m <= N. */
int lbm_get_populations_at(lbm_t* ctx, const int32_t* cells, int m, void* f);
/* Load populations (same format); resets the AA parity to even. */
int lbm_set_populations(lbm_t* ctx, const void* f);

/* Introspection used by the harness: number of time steps done; number of fluid cells; bytes of
 * device memory held; number of kernels launched by this context so far. */
long long lbm_steps_done(const lbm_t* ctx);
long long lbm_num_fluid(const lbm_t* ctx);
long long lbm_device_bytes(const lbm_t* ctx);
long long lbm_kernel_launches(const lbm_t* ctx);
/* Block until everything queued on the context's stream has finished. */
int lbm_sync(lbm_t* ctx);
/* Select an implementation variant of the step kernels; results are identical across variants
 * (tests compare them bit for bit).  0 default (library's choice); 1 generic_push: two-population as
 * the paper's collide-then-push (Table 1); 2 generic_pull: as pull-then-collide with
 * lazily streamed storage (the default); 3 aos_plain: AoS without the shared-memory tile; 4 tma: SoA
 * loads staged through shared memory by TMA bulk copies; 5 no_tma: never that kernel; 6 plain:
 * one cell per thread, no L2 prefetch, no programmatic dependent launch, every kernel walks the cells upwards
 * (by default successive kernels alternate the direction to reuse what the last one left in L2); 7 aos_march: AoS
 * two-population pull with the neighbour records in a marching shared-memory tile (only when the
 * outermost x-layers hold no fluid or ghost cell; otherwise the default kernels run).  Variants 4
 * and 7 are measured alternatives that lose to the default.  Unknown: LBM_E_ARG. */
int lbm_set_variant(lbm_t* ctx, int variant);

/* Threads per block of the step kernels (tuning knob of the sweep; multiple of 32 in [32, 256];
 * default 128).  Results do not depend on it. */
int lbm_set_block(lbm_t* ctx, int threads);

/* Slab decomposition along x (the slowest axis: an x-layer is ny*nz contiguous cells of every SoA
 * plane).  The paper's scheme is single-device; cells are coupled only through the
 * one-cell stencil of Eq 2, so a rank owns the layers x = 1 .. nx-2 of its context
 * and flags x = 0 and x = nx-1 LBM_GHOST (or WALL/MOVING where the neighbouring rank's layer is
 * solid).  SoA schemes only (two-population in its pull form, swap, AA); LBM_E_ARG otherwise, and
 * lbm_set_flags refuses LBM_GHOST cells there.
 *
 * One time step in parts, so that the halo travels while the bulk of the slab is updated:
 *   lbm_step_begin    the step's kernel on the outermost owned layers x = 1 and x = nx-2 only
 *                     (swap: pass 1).  Layers 0 and nx-1 are never updated: LBM_E_STATE if they
 *                     hold a FLUID cell;
 *   lbm_halo_pack     (both faces) buf <- what leaves through the face; start the transfer;
 *   lbm_step_end      the same kernel on the layers 2 .. nx-3;
 *   lbm_halo_unpack   (both faces) once the neighbours' buffers have arrived;
 *   lbm_step_finish   completes the step (swap: pass 2, which needs the halo).
 * Between begin and finish no other call on the context is allowed (LBM_E_STATE).  The result is
 * bit for bit that of the undivided lattice.  What a message holds depends on the scheme (Table 1,
 * PAPER.md:L147-159; 5 of 19 or 9 of 27 directions per face, those with c_x pointing out of it, in
 * increasing k, layout [dir][ny*nz], raw stored values of the context dtype):
 *   two-population   post-collision f_out_k of the outermost owned layer (slot k); unpack writes
 *                    the ghost layer, from which the next step pulls;
 *   AA, even step    the same values, which this step keeps in slot kbar; unpack writes the ghost
 *                    layer ("AA exchanges on odd steps only": the odd step pulls them from there);
 *   AA, odd step     the odd step pushes into slot k of x + c_k, i.e. into the ghost layer: pack
 *                    reads the ghost layer, unpack merges into the neighbour's outermost owned
 *                    layer, skipping cells whose upstream cell is solid (they bounced back);
 *   swap             after pass 1 (as AA even); through the low face the ghost layer is written,
 *                    through the high face the half of the pass-2 exchange that the (absent) thread
 *                    of the ghost cell would have done is applied on arrival.
 * A context with GHOST cells stepped by plain lbm_step(1) (two-population, AA) needs pack / unpack
 * after every step; lbm_step(n > 1) and the swap scheme return LBM_E_STATE there.
 * buf is DEVICE memory of lbm_halo_count() elements; every call is asynchronous on the stream. */
int lbm_step_begin(lbm_t* ctx);
int lbm_step_end(lbm_t* ctx);
int lbm_step_finish(lbm_t* ctx);
long long lbm_halo_count(const lbm_t* ctx);
int lbm_halo_pack(lbm_t* ctx, int face, void* buf_dev);
int lbm_halo_unpack(lbm_t* ctx, int face, const void* buf_dev);

/* The same step driven inside the library, the halo stored by the pack kernel straight into the
 * neighbouring slab's receive buffer (peer memory: NVLink between GPUs) and a sequence number
 * published behind it; the neighbour's unpack kernel waits for that number (bounded).  No host
 * code runs between the parts and nothing goes through a communication library.
 *   lbm_slab_link(ctx, face, peer)   the slab beyond `face` is context `peer` of this process (any
 *                                    device with peer access; peer == ctx closes a periodic ring of
 *                                    one slab; NULL = nothing beyond: that face is never exchanged);
 *   lbm_slab_export / lbm_slab_import   the same across processes through a 64-byte CUDA IPC
 *                                    handle of the receive block (export mine, import the
 *                                    neighbour's for `face`); same ny, nz, lattice, scheme, dtype;
 *   lbm_slab_post      lbm_step_begin, both peer stores, lbm_step_end;
 *   lbm_slab_complete  both merges, lbm_step_finish;
 *   lbm_slab_step(n)   n times post + complete (every slab on its own device and stream).  Several
 *                      slabs on ONE stream must alternate instead: post on all, then complete on all;
 *   lbm_slab_status    LBM_E_STATE if some message never arrived (synchronises).
 * A context lives on the CUDA device that was current at lbm_create, and every call on it expects that
 * device to be current; lbm_slab_link / post / complete / step switch to it themselves, so one host
 * thread can drive the slabs of several GPUs. */
int lbm_slab_link(lbm_t* ctx, int face, lbm_t* peer);
int lbm_slab_export(lbm_t* ctx, void* handle64);
int lbm_slab_import(lbm_t* ctx, int face, const void* handle64);
int lbm_slab_post(lbm_t* ctx);
int lbm_slab_complete(lbm_t* ctx);
int lbm_slab_step(lbm_t* ctx, int n);
int lbm_slab_status(lbm_t* ctx);

/* CUDA-graph replay of lbm_step.  A step of a small lattice lasts a few microseconds and is bound
 * by launch latency (the paper's "one synchronisation per step"), and up to ~128^3
 * the gaps between launches still cost 2-5 %; lbm_step(n) then captures 16 steps once and replays
 * the graph.  LBM_GRAPH_AUTO (default): lattices of at most 160^3 cells; LBM_GRAPH_OFF: never;
 * LBM_GRAPH_ON: any size.  Results are identical (same kernels, same order).  lbm_graph_replays =
 * graph launches so far. */
enum { LBM_GRAPH_AUTO = 0, LBM_GRAPH_OFF = 1, LBM_GRAPH_ON = 2 };
int lbm_set_graph(lbm_t* ctx, int mode);
long long lbm_graph_replays(const lbm_t* ctx);

const char* lbm_last_error(void);
const char* lbm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
