// lbm_api.cu -- the C ABI of include/lbm.h: context, state machine of the schemes, argument
// checks and kernel launches.  No arithmetic of the method lives here; every step of the path
// runs in the kernels of kernels.cuh / collision.cuh / aux.cu.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/lbm.h"
#include "dispatch.cuh"

using namespace lbm;

namespace {

thread_local char g_err[512] = "";
void set_err(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

lbm_alloc_fn g_alloc = nullptr;
lbm_free_fn g_free = nullptr;
cudaStream_t g_stream = nullptr;

enum Family { FAM_2POP, FAM_SWAP, FAM_AA };
// what the halo calls of a slab decomposition move after the step part that ran last (lbm_halo_pack)
enum HaloMode {
    HALO_NONE,
    HALO_POST_K,     // post-collision value of direction k in slot k of its own cell (two-population pull form)
    HALO_POST_KBAR,  // ... in slot kbar of its own cell (AA even step, swap pass 1)
    HALO_PUSHED      // AA odd step: slot k of the cell at x + c_k, i.e. in the ghost layer
};
// where the pre-collision state of the current time lives
enum Storage {
    STO_NONE,      // nothing loaded yet
    STO_CANON,     // pop_k(x) = f_k(x)                      (LD_LOCAL)
    STO_POST,      // pop holds f_out of the previous step   (LD_PULL), 2-pop pull form
    STO_AA_ODD     // after an AA even step                  (LD_AAPULL)
};

}  // namespace

struct lbm_ctx {
    int nx, ny, nz, Q, model, scheme, dtype;
    int device;         // CUDA device that was current at lbm_create: every buffer and the stream live there
    Family fam;
    bool soa;
    double omega, omega_bulk, omega3, omega_hi, trt_magic;
    double u_wall[3];
    Geo g;
    size_t elem;        // bytes per population
    size_t pop_elems;   // elements in one population array
    void* pop[2];       // [1] only for FAM_2POP
    void* pop_first;    // pop[0] as allocated: tells the parity of the two-population pointer exchange
    uint8_t* code;
    uint2* grp;                // per 32 cells: ordinal of the first edge cell, bit set of edge cells (kernels.cuh)
    unsigned long long* mask;  // link masks of the edge cells only, [n_edge]
    long long n_edge;
    void* scratch;      // 4 planes of N elements (rho,u staging; plane import/export): held only while a
    size_t scratch_bytes;  // host-facing call runs (scratch_get / scratch_release)
    bool outer_fluid, has_ghost;   // flags: FLUID in x-layer 0 or nx-1; any GHOST cell
    double* partial;    // energy partial sums
    double* e_dev;
    int n_partial;
    Storage sto;
    int variant;
    int block;
    long long steps, launches, dev_bytes, n_fluid;
    lbm_alloc_fn alloc;
    lbm_free_fn free_fn;
    cudaStream_t stream;
    int c[27][3], opp[27];
    int sslot[27];   // storage slot of direction k: k in SoA, its place inside the record in AoS (lattice.cuh)
    double w[27];
    // CUDA-graph replay of lbm_step for launch-bound lattices (see step_graphed)
    int graph_mode;             // LBM_GRAPH_AUTO / OFF / ON
    cudaGraphExec_t graph_exec[2]; // GRAPH_STEPS steps starting from graph_sto[j] with pop[0] == graph_pop0[j]: one per
                                   // parity, so that lbm_step(17) called repeatedly does not re-capture every time
    int prefetch;                // L2 prefetch distance of the step kernels in cells, -1 = the tuned distances, 0 = off (variant "plain")
    int pdl;                     // programmatic dependent launch of the step kernels (off in variant "plain")
    int range_first, range_end;  // cells the next step launch covers (0, 0 = all); lbm_step_begin / lbm_step_end
    int mid_step;                // 0, 1 after lbm_step_begin, 2 after lbm_step_end (until lbm_step_finish)
    int halo_mode;               // HaloMode
    // slab driver (lbm_slab_post / lbm_slab_complete): my receive buffers, flags and counters, and
    // the same block of the slab beyond each face (this process: lbm_slab_link; another: CUDA IPC)
    char* slab_mem;
    char* peer_mem[2];
    bool peer_ipc[2];
    unsigned long long seq_out[2], seq_in[2];
    cudaStream_t cap_stream;    // private stream the capture runs on (the context stream may be the
                                // legacy default stream, which cannot be captured); nothing executes on it
    Storage graph_sto[2];
    void* graph_pop0[2];
    int graph_next;             // slot the next capture replaces
    long long graph_replays;
};

namespace {

void* dev_alloc(lbm_ctx* c, size_t bytes)
{
    void* p = nullptr;
    if (c->alloc) p = c->alloc(bytes);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) p = nullptr;
    if (p) c->dev_bytes += (long long)bytes;
    return p;
}
void dev_free(lbm_ctx* c, void* p, size_t bytes = 0)
{
    if (!p) return;
    c->dev_bytes -= (long long)bytes;
    if (c->free_fn) c->free_fn(p);
    else cudaFree(p);
}

// the staging area of the host-facing calls (flag upload, rho/u staging, plane import/export) is
// allocated when such a call starts and released when it ends (they all synchronise), so that a
// context at rest holds the populations, 1.25 B per cell of codes and the masks of the edge cells
void* scratch_get(lbm_ctx* c, size_t bytes)
{
    if (c->scratch && c->scratch_bytes >= bytes) return c->scratch;
    if (c->scratch) { dev_free(c, c->scratch, c->scratch_bytes); c->scratch = nullptr; c->scratch_bytes = 0; }
    c->scratch = dev_alloc(c, bytes);
    if (c->scratch) c->scratch_bytes = bytes;
    return c->scratch;
}
// call only after the stream has been synchronised
void scratch_release(lbm_ctx* c)
{
    if (c->scratch) dev_free(c, c->scratch, c->scratch_bytes);
    c->scratch = nullptr;
    c->scratch_bytes = 0;
}

int cuda_fail(const char* what, cudaError_t e)
{
    set_err("%s: %s", what, cudaGetErrorString(e));
    return LBM_E_CUDA;
}
#define CK(call)                                         \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) return cuda_fail(#call, e_); \
    } while (0)

// load / store modes of a step-kernel kind (kernels.cuh)
void kind_modes(int kind, int* load, int* store)
{
    switch (kind) {
    case SK_PUSH: *load = LD_LOCAL; *store = ST_PUSH; break;
    case SK_PULL: *load = LD_PULL; *store = ST_LOCAL; break;
    case SK_COLLIDE: *load = LD_LOCAL; *store = ST_LOCAL; break;
    case SK_EVEN: *load = LD_LOCAL; *store = ST_SWAPPED; break;
    default: *load = LD_AAPULL; *store = ST_PUSH; break;
    }
}

template <class T>
StepArgs<T> make_args(const lbm_ctx* c, const void* src, void* dst, int load = LD_LOCAL, int store = ST_LOCAL)
{
    StepArgs<T> a;
    const long long is = c->soa ? 1 : c->Q;  // elements per cell step
    for (int k = 0; k < 27; ++k) {
        a.plane[k] = a.ldo[k] = a.sto[k] = a.wlo[k] = a.wso[k] = 0;
        if (k >= c->Q) continue;
        const int kb = c->opp[k];
        const long long off = ((long long)c->c[k][0] * c->ny + c->c[k][1]) * c->nz + c->c[k][2];
        const long long pk = c->soa ? (long long)k * c->g.stride : c->sslot[k];
        const long long pkb = c->soa ? (long long)kb * c->g.stride : c->sslot[kb];
        a.plane[k] = pk;
        a.ldo[k] = (long long)sizeof(T) * (load == LD_LOCAL ? pk : load == LD_PULL ? pk - off * is : pkb - off * is);
        a.sto[k] = (long long)sizeof(T) * (store == ST_LOCAL ? pk : store == ST_SWAPPED ? pkb : pk + off * is);
        a.wlo[k] = (long long)sizeof(T) * (load == LD_PULL ? pkb : pk);
        a.wso[k] = (long long)sizeof(T) * pkb;
    }
    a.src = (const T*)src;
    a.dst = (T*)dst;
    for (int k = 0; k < 27; ++k) {
        a.lp[k] = a.src ? a.src + a.ldo[k] / (long long)sizeof(T) : nullptr;
        a.sp[k] = a.dst ? a.dst + a.sto[k] / (long long)sizeof(T) : nullptr;
    }
    a.code = c->code;
    a.grp = c->grp;
    a.mask = c->mask;
    a.g = c->g;
    a.pdl = c->pdl;
    a.pf = 0;
    a.pf_strided = 0;
    a.tma = 0;
    a.rev = 0;
    a.march = !c->soa && !c->outer_fluid && !c->has_ghost && c->variant == V_AOS_MARCH;
    a.patch = !c->soa && c->variant == V_DEFAULT && c->ny <= 65535 && c->nx <= 65535;   // grid.y / grid.z limits
    a.first = c->range_first;
    a.end = c->range_end > 0 ? c->range_end : c->g.n;
    a.rt.omega = (T)c->omega;
    a.rt.omega_bulk = (T)c->omega_bulk;
    a.rt.omega3 = (T)c->omega3;
    a.rt.omega_hi = (T)c->omega_hi;
    // TRT: Lambda = (1/w+ - 1/2)(1/w- - 1/2)
    a.rt.omega_minus = (T)(1.0 / (c->trt_magic / (1.0 / c->omega - 0.5) + 0.5));
    for (int k = 0; k < 27; ++k) {
        double cu = 0.0;
        if (k < c->Q) cu = c->c[k][0] * c->u_wall[0] + c->c[k][1] * c->u_wall[1] + c->c[k][2] * c->u_wall[2];
        a.wterm[k] = k < c->Q ? (T)(-6.0 * c->w[k] * cu) : (T)0;  // Eq 3, rho_w = 1
    }
    return a;
}

template <class T, int Q>
cudaError_t step_model(const lbm_ctx* c, int kind, const StepArgs<T>& a)
{
    const bool soa = c->soa;
    const bool st = c->variant != V_AOS_PLAIN;
    const int b = c->block;
    cudaStream_t s = c->stream;
    switch (c->model) {
    case LBM_BGK_W2: return launch_step<T, Q, M_BGK_W2>(kind, soa, b, st, a, s);
    case LBM_TRT: return launch_step<T, Q, M_TRT>(kind, soa, b, st, a, s);
    case LBM_REG: return launch_step<T, Q, M_REG>(kind, soa, b, st, a, s);
    default: break;
    }
    // every moment of order >= 3 relaxed with exactly 1: the variant that never computes their
    // pre-collision values (collision.cuh).  Same result up to round-off.
    if (c->omega3 == 1.0 && c->omega_hi == 1.0) {
        switch (c->model) {
        case LBM_RM: return launch_step<T, Q, M_RM_E>(kind, soa, b, st, a, s);
        case LBM_HM: return launch_step<T, Q, M_HM_E>(kind, soa, b, st, a, s);
        case LBM_CM: return launch_step<T, Q, M_CM_E>(kind, soa, b, st, a, s);
        case LBM_CHM: return launch_step<T, Q, M_CHM_E>(kind, soa, b, st, a, s);
        case LBM_K: return launch_step<T, Q, M_K_E>(kind, soa, b, st, a, s);
        default: break;
        }
    }
    {
        switch (c->model) {
        case LBM_BGK_NW4: return launch_step<T, Q, M_BGK_NW4>(kind, soa, b, st, a, s);
        case LBM_RM: return launch_step<T, Q, M_RM>(kind, soa, b, st, a, s);
        case LBM_HM: return launch_step<T, Q, M_HM>(kind, soa, b, st, a, s);
        case LBM_CM: return launch_step<T, Q, M_CM>(kind, soa, b, st, a, s);
        case LBM_CHM: return launch_step<T, Q, M_CHM>(kind, soa, b, st, a, s);
        case LBM_K: return launch_step<T, Q, M_K>(kind, soa, b, st, a, s);
        case LBM_RR: return launch_step<T, Q, M_RR>(kind, soa, b, st, a, s);
        default: break;
        }
    }
    return cudaErrorInvalidValue;
}

// the alternating direction pays as soon as the populations do not fit in L2 as a whole (below that every
// line hits anyway)
bool beyond_l2_half(const lbm_ctx* c) { return c->pop_elems * c->elem * (c->fam == FAM_2POP ? 2 : 1) > (size_t)60 << 20; }

template <class T>
cudaError_t step_kind(lbm_ctx* c, int kind, const void* src, void* dst)
{
    int load, store;
    kind_modes(kind, &load, &store);
    StepArgs<T> a = make_args<T>(c, src, dst, load, store);
    // L2 prefetch ahead of the block scheduler (kernels.cuh) for the kernels of the steady state: per
    // thread in fp64, one warp in 32 with a line per lane in fp32; nothing when the populations fit
    // in L2 anyway (48^3: -5 %, 64^3: -3 % with it).  The variant "plain" switches it off.
    const bool beyond_l2 = c->pop_elems * c->elem * (c->fam == FAM_2POP ? 2 : 1) > (size_t)100 << 20;
    if (c->soa && beyond_l2 && (kind == SK_EVEN || kind == SK_ODD || kind == SK_PULL)) {
        a.pf_strided = sizeof(T) == 4;
        a.pf = c->prefetch >= 0 ? c->prefetch : (sizeof(T) == 4 ? 65536 : 16384);
    }
    // successive step kernels walk the lattice in alternating directions, so that each starts on the lines its
    // predecessor left in L2 (kernels.cuh): a pure function of the storage state, hence the same inside a
    // captured graph.  SoA launches, the whole lattice or a range of x-layers (slab steps: the interior
    // range is nearly the whole slab); variant "plain" walks upwards always.
    if (c->soa && beyond_l2_half(c) && c->variant != V_PLAIN && c->variant != V_TMA) {
        a.rev = kind == SK_ODD ? 1 : kind == SK_PULL ? (c->pop[0] != c->pop_first) : 0;
        if (a.rev) a.pf = -a.pf;
    }
    if (c->soa && c->variant == V_TMA) { a.tma = 1; a.pf = 0; }
    c->launches++;
    return c->Q == 19 ? step_model<T, 19>(c, kind, a) : step_model<T, 27>(c, kind, a);
}
cudaError_t step_kind(lbm_ctx* c, int kind, const void* src, void* dst)
{
    return c->dtype == LBM_F64 ? step_kind<double>(c, kind, src, dst) : step_kind<float>(c, kind, src, dst);
}

int load_mode(const lbm_ctx* c)
{
    return c->sto == STO_POST ? LD_PULL : c->sto == STO_AA_ODD ? LD_AAPULL : LD_LOCAL;
}

// the pull form is the default for 2-pop: aligned stores, measured faster on B200
bool use_pull(const lbm_ctx* c) { return c->variant != V_GENERIC_PUSH; }

// bring post-collision 2-pop storage back to canonical (one stream-only pass)
int normalise(lbm_ctx* c)
{
    if (c->sto != STO_POST) return LBM_OK;
    cudaError_t e;
    if (c->dtype == LBM_F64) e = aux_stream_only<double>(c->Q, c->soa, make_args<double>(c, c->pop[0], c->pop[1], LD_PULL, ST_LOCAL), c->stream);
    else e = aux_stream_only<float>(c->Q, c->soa, make_args<float>(c, c->pop[0], c->pop[1], LD_PULL, ST_LOCAL), c->stream);
    c->launches++;
    if (e != cudaSuccess) return cuda_fail("stream_only", e);
    void* t = c->pop[0]; c->pop[0] = c->pop[1]; c->pop[1] = t;
    c->sto = STO_CANON;
    return LBM_OK;
}

// swap pass 2 over every cell (Table 1)
int swap_pass2(lbm_ctx* c)
{
    const bool pf = c->soa && c->pop_elems * c->elem > (size_t)100 << 20;  // as in step_kind
    const bool rev = c->soa && beyond_l2_half(c) && c->variant != V_PLAIN;   // pass 1 walks upwards, pass 2 downwards (step_kind)
    if (c->dtype == LBM_F64) {
        StepArgs<double> a = make_args<double>(c, c->pop[0], c->pop[0]);
        if (pf) a.pf = c->prefetch >= 0 ? c->prefetch : 16384;
        if (rev) { a.rev = 1; a.pf = -a.pf; }
        CK(aux_swap_stream<double>(c->Q, c->soa, a, c->stream));
    } else {
        StepArgs<float> a = make_args<float>(c, c->pop[0], c->pop[0]);
        if (pf) { a.pf = c->prefetch >= 0 ? c->prefetch : 65536; a.pf_strided = 1; }
        if (rev) { a.rev = 1; a.pf = -a.pf; }
        CK(aux_swap_stream<float>(c->Q, c->soa, a, c->stream));
    }
    c->launches++;
    return LBM_OK;
}

// one collide-and-stream cycle by the context's scheme (Table 1)
int one_step(lbm_ctx* c)
{
    if (c->fam == FAM_2POP) {
        if (use_pull(c)) {
            if (c->sto == STO_CANON) {  // (S C)^n = S (C S)^(n-1) C: start with a collide-only pass
                CK(step_kind(c, SK_COLLIDE, c->pop[0], c->pop[0]));
                c->sto = STO_POST;
            } else {
                CK(step_kind(c, SK_PULL, c->pop[0], c->pop[1]));
                void* t = c->pop[0]; c->pop[0] = c->pop[1]; c->pop[1] = t;
            }
        } else {
            if (int rc = normalise(c)) return rc;
            CK(step_kind(c, SK_PUSH, c->pop[0], c->pop[1]));
            void* t = c->pop[0]; c->pop[0] = c->pop[1]; c->pop[1] = t;
        }
    } else if (c->fam == FAM_AA) {
        if (c->sto == STO_CANON) {
            CK(step_kind(c, SK_EVEN, c->pop[0], c->pop[0]));
            c->sto = STO_AA_ODD;
        } else {
            CK(step_kind(c, SK_ODD, c->pop[0], c->pop[0]));
            c->sto = STO_CANON;
        }
    } else {
        CK(step_kind(c, SK_EVEN, c->pop[0], c->pop[0]));  // pass 1: collide into opposite slots
        if (int rc = swap_pass2(c)) return rc;
    }
    c->halo_mode = c->fam == FAM_SWAP ? HALO_NONE
                 : c->fam == FAM_2POP ? (use_pull(c) ? HALO_POST_K : HALO_NONE)
                 : c->sto == STO_AA_ODD ? HALO_POST_KBAR : HALO_PUSHED;
    c->steps++;
    return LBM_OK;
}

// ---- CUDA-graph replay.  Below ~64^3 cells a step kernel runs for a few microseconds and the
// time step is bound by launch latency (one launch per step, two for swap; "one
// synchronisation per step").  GRAPH_STEPS steps are captured once into a graph (kernel arguments
// baked in) and replayed; every scheme returns to the same storage state and the same pop[0]
// after an even number of steps, so one graph serves the whole run.  Any call that changes what
// the kernels would be given (rates, flags, variant, block, populations' home) drops the graph.
enum { GRAPH_STEPS = 16, GRAPH_AUTO_MAX_CELLS = 160 * 160 * 160 };

void drop_graph(lbm_ctx* c)
{
    for (int j = 0; j < 2; ++j) {
        if (c->graph_exec[j]) cudaGraphExecDestroy(c->graph_exec[j]);
        c->graph_exec[j] = nullptr;
    }
}

bool graph_wanted(const lbm_ctx* c, int n)
{
    if (n < GRAPH_STEPS || c->graph_mode == LBM_GRAPH_OFF) return false;
    return c->graph_mode == LBM_GRAPH_ON || c->g.n <= GRAPH_AUTO_MAX_CELLS;
}

// run GRAPH_STEPS steps through the cached graph (capturing it first if needed)
int step_graphed(lbm_ctx* c)
{
    if (c->fam == FAM_2POP && use_pull(c) && c->sto == STO_CANON) return LBM_E_STATE;  // first step differs from the rest
    int slot = -1;
    for (int j = 0; j < 2; ++j)
        if (c->graph_exec[j] && c->graph_sto[j] == c->sto && c->graph_pop0[j] == c->pop[0]) slot = j;
    if (slot < 0) {
        slot = !c->graph_exec[0] ? 0 : !c->graph_exec[1] ? 1 : c->graph_next;
        c->graph_next = 1 - slot;
        if (c->graph_exec[slot]) { cudaGraphExecDestroy(c->graph_exec[slot]); c->graph_exec[slot] = nullptr; }
        cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
        if (c->stream != nullptr && c->stream != cudaStreamLegacy && c->stream != cudaStreamPerThread &&
            (cudaStreamIsCapturing(c->stream, &st) != cudaSuccess || st != cudaStreamCaptureStatusNone)) {
            cudaGetLastError();
            return LBM_E_STATE;  // the caller is capturing this stream itself
        }
        if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
            c->cap_stream = nullptr;
            cudaGetLastError();
            return LBM_E_STATE;
        }
        const Storage sto0 = c->sto;
        const int halo0 = c->halo_mode;
        void* const pop0 = c->pop[0];
        const long long steps0 = c->steps, launches0 = c->launches;
        cudaStream_t const user_stream = c->stream;
        if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return LBM_E_STATE; }
        c->stream = c->cap_stream;
        int rc = LBM_OK;
        for (int s = 0; s < GRAPH_STEPS && rc == LBM_OK; ++s) rc = one_step(c);
        c->stream = user_stream;
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
        // nothing ran: undo the bookkeeping of the captured steps
        c->steps = steps0; c->launches = launches0;
        const bool periodic = c->sto == sto0 && c->pop[0] == pop0;
        c->sto = sto0;
        c->halo_mode = halo0;
        if (c->pop[0] != pop0) { void* t = c->pop[0]; c->pop[0] = c->pop[1]; c->pop[1] = t; }
        if (rc != LBM_OK || e != cudaSuccess || !graph || !periodic) {
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            return LBM_E_STATE;
        }
        e = cudaGraphInstantiate(&c->graph_exec[slot], graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) { c->graph_exec[slot] = nullptr; cudaGetLastError(); return LBM_E_STATE; }
        c->graph_sto[slot] = sto0;
        c->graph_pop0[slot] = pop0;
    }
    CK(cudaGraphLaunch(c->graph_exec[slot], c->stream));
    c->steps += GRAPH_STEPS;
    c->launches += GRAPH_STEPS * (c->fam == FAM_SWAP ? 2 : 1);
    c->graph_replays++;
    return LBM_OK;
}

// cell codes, group table and compact link masks from N flag bytes in device memory (kernels.cuh);
// synchronises (the number of edge cells sizes the mask array)
int classify(lbm_ctx* c, const uint8_t* flags_dev)
{
    // the energy partials (n/256 doubles) double as scratch here: one unsigned for the total, then the
    // block sums of the prefix scan (n/32768 unsigned)
    unsigned* total = reinterpret_cast<unsigned*>(c->partial);
    CK(aux_classify_codes(c->Q, flags_dev, c->code, c->grp, total, total + 4, c->g, c->stream));
    unsigned n_edge = 0;
    CK(cudaMemcpyAsync(&n_edge, total, sizeof n_edge, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (c->mask) dev_free(c, c->mask, sizeof(unsigned long long) * (size_t)(c->n_edge > 0 ? c->n_edge : 1));
    c->n_edge = n_edge;
    c->mask = (unsigned long long*)dev_alloc(c, sizeof(unsigned long long) * (size_t)(n_edge > 0 ? n_edge : 1));
    if (!c->mask) { set_err("device allocation failed (link masks of %u edge cells)", n_edge); return LBM_E_ALLOC; }
    CK(aux_classify_masks(c->Q, flags_dev, c->code, c->grp, c->mask, c->g, c->stream));
    c->launches += 5;
    CK(cudaStreamSynchronize(c->stream));
    return LBM_OK;
}

}  // namespace

extern "C" {

const char* lbm_last_error(void) { return g_err; }
const char* lbm_version(void) { return "lbm_b200 0.1 (sm_100a)"; }

int lbm_set_hooks(lbm_alloc_fn alloc, lbm_free_fn free_fn, void* stream)
{
    if ((alloc == nullptr) != (free_fn == nullptr)) { set_err("alloc and free hooks must be given together"); return LBM_E_ARG; }
    g_alloc = alloc;
    g_free = free_fn;
    g_stream = (cudaStream_t)stream;
    return LBM_OK;
}

lbm_t* lbm_create(int nx, int ny, int nz, int lattice, int collision, int scheme, double omega, int dtype)
{
    if (nx < 3 || ny < 3 || nz < 3) { set_err("extents must be >= 3 (got %d %d %d)", nx, ny, nz); return nullptr; }
    if ((long long)nx * ny * nz >= (1LL << 31) - 1024) { set_err("too many cells"); return nullptr; }  // cell indices, rounded up to a block, stay in int
    if (lattice != LBM_D3Q19 && lattice != LBM_D3Q27) { set_err("lattice must be 19 or 27"); return nullptr; }
    if (collision < 0 || collision >= LBM_NUM_MODELS) { set_err("unknown collision model %d", collision); return nullptr; }
    if (scheme < 0 || scheme >= LBM_NUM_SCHEMES) { set_err("unknown scheme %d", scheme); return nullptr; }
    if (dtype != LBM_F32 && dtype != LBM_F64) { set_err("dtype must be LBM_F32 or LBM_F64"); return nullptr; }
    if (!(omega > 0.0 && omega < 2.0)) { set_err("omega must be in (0,2)"); return nullptr; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        set_err("no CUDA device: this library has no CPU fallback");
        return nullptr;
    }
    lbm_ctx* c = new (std::nothrow) lbm_ctx();
    if (!c) { set_err("out of host memory"); return nullptr; }
    memset(c, 0, sizeof *c);
    cudaGetDevice(&c->device);
    c->nx = nx; c->ny = ny; c->nz = nz; c->Q = lattice; c->model = collision; c->scheme = scheme; c->dtype = dtype;
    c->fam = (scheme == LBM_2POP_SOA || scheme == LBM_2POP_AOS) ? FAM_2POP
           : (scheme == LBM_SWAP_SOA || scheme == LBM_SWAP_AOS) ? FAM_SWAP : FAM_AA;
    c->soa = scheme == LBM_2POP_SOA || scheme == LBM_SWAP_SOA || scheme == LBM_AA_SOA;
    c->omega = omega;
    c->omega_bulk = omega;                                   // R14
    c->omega3 = collision == LBM_RR ? omega : 1.0;           // R14
    c->omega_hi = collision == LBM_RR ? omega : 1.0;
    c->trt_magic = 0.25;                                     // R15
    c->elem = dtype == LBM_F64 ? 8 : 4;
    c->g.nx = nx; c->g.ny = ny; c->g.nz = nz; c->g.n = nx * ny * nz;
    const long long per128 = 128 / (long long)c->elem;
    c->g.stride = ((long long)c->g.n + per128 - 1) / per128 * per128;  // planes start 128 B aligned
    c->pop_elems = c->soa ? (size_t)c->g.stride * c->Q : (size_t)c->g.n * c->Q;
    c->alloc = g_alloc; c->free_fn = g_free; c->stream = g_stream;
    c->variant = V_DEFAULT;
    c->pdl = 1;
    c->prefetch = -1;
    c->block = 128;
    c->n_fluid = c->g.n;
    lattice_tables(c->Q, c->c, c->opp, c->w, c->sslot);
    if (c->soa) for (int k = 0; k < c->Q; ++k) c->sslot[k] = k;

    const int narr = c->fam == FAM_2POP ? 2 : 1;
    bool ok = true;
    for (int a = 0; a < narr && ok; ++a) {
        c->pop[a] = dev_alloc(c, c->pop_elems * c->elem);
        if (a == 0) c->pop_first = c->pop[0];
        ok = c->pop[a] != nullptr;
        if (ok) ok = cudaMemsetAsync(c->pop[a], 0, c->pop_elems * c->elem, c->stream) == cudaSuccess;
    }
    if (ok) { c->code = (uint8_t*)dev_alloc(c, (size_t)c->g.n); ok = c->code != nullptr; }
    if (ok) ok = cudaMemsetAsync(c->code, 0, (size_t)c->g.n, c->stream) == cudaSuccess;
    if (ok) { c->grp = (uint2*)dev_alloc(c, sizeof(uint2) * (size_t)((c->g.n + 31) / 32)); ok = c->grp != nullptr; }
    c->n_partial = (c->g.n + 255) / 256;  // one partial per block of 256 cells, then two fixed summing stages
    if (ok) { c->partial = (double*)dev_alloc(c, sizeof(double) * (c->n_partial + ENERGY_STAGE2 + 1)); ok = c->partial != nullptr; }
    if (!ok) {
        set_err("device allocation failed (%lld bytes so far): %s", c->dev_bytes, cudaGetErrorString(cudaGetLastError()));
        lbm_destroy(c);
        return nullptr;
    }
    c->e_dev = c->partial + c->n_partial + ENERGY_STAGE2;
    // cells on the faces of a fully periodic box still need the wrap: classify with all-fluid flags
    void* zero = scratch_get(c, (size_t)c->g.n);
    if (!zero || cudaMemsetAsync(zero, 0, (size_t)c->g.n, c->stream) != cudaSuccess || classify(c, (const uint8_t*)zero) != LBM_OK) {
        if (!zero) set_err("device allocation failed (%lld bytes so far)", c->dev_bytes);
        lbm_destroy(c);
        return nullptr;
    }
    scratch_release(c);
    c->outer_fluid = true;
    c->has_ghost = false;
    return c;
}

int lbm_destroy(lbm_t* c)
{
    if (!c) return LBM_OK;
    cudaStreamSynchronize(c->stream);
    drop_graph(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    dev_free(c, c->pop[0]);
    dev_free(c, c->pop[1]);
    dev_free(c, c->code);
    dev_free(c, c->grp);
    dev_free(c, c->mask);
    dev_free(c, c->scratch);
    dev_free(c, c->partial);
    for (int f = 0; f < 2; ++f)
        if (c->peer_ipc[f] && c->peer_mem[f]) cudaIpcCloseMemHandle(c->peer_mem[f]);
    if (c->slab_mem) cudaFree(c->slab_mem);
    delete c;
    return LBM_OK;
}

int lbm_set_flags(lbm_t* c, const uint8_t* flags, const double u_wall[3])
{
    if (!c || !flags) { set_err("null argument"); return LBM_E_ARG; }
    long long nfluid = 0;
    bool ghost = false, outer = false;
    const long long layer = (long long)c->ny * c->nz;
    for (long long i = 0; i < c->g.n; ++i) {
        if (flags[i] > LBM_GHOST) { set_err("flag %d at cell %lld is not FLUID/WALL/MOVING/GHOST", flags[i], i); return LBM_E_ARG; }
        nfluid += flags[i] == LBM_FLUID;
        ghost |= flags[i] == LBM_GHOST;
        outer |= flags[i] == LBM_FLUID && (i < layer || i >= c->g.n - layer);
    }
    // ghost cells are filled by the halo calls, which exist for the SoA layouts only (and not for the
    // paper's push form of the two-population scheme): anywhere else their populations would be lost
    if (ghost && (!c->soa || c->variant == V_GENERIC_PUSH)) {
        set_err("LBM_GHOST cells need a halo exchange: SoA schemes only (not AoS, not the generic_push variant)");
        return LBM_E_ARG;
    }
    drop_graph(c);
    for (int a = 0; a < 3; ++a) c->u_wall[a] = u_wall ? u_wall[a] : 0.0;
    void* stage = scratch_get(c, (size_t)c->g.n);
    if (!stage) { set_err("device allocation failed (flag staging)"); return LBM_E_ALLOC; }
    CK(cudaMemcpyAsync(stage, flags, (size_t)c->g.n, cudaMemcpyHostToDevice, c->stream));
    if (int rc = classify(c, (const uint8_t*)stage)) return rc;
    scratch_release(c);
    c->n_fluid = nfluid;
    c->has_ghost = ghost;
    c->outer_fluid = outer;
    c->sto = STO_NONE;  // populations of cells that changed type are meaningless now
    c->mid_step = 0;
    c->halo_mode = HALO_NONE;
    return LBM_OK;
}

#define NOT_MID_STEP(c, what) \
    do { if ((c)->mid_step) { set_err(what " between lbm_step_begin and lbm_step_finish"); return LBM_E_STATE; } } while (0)

int lbm_set_relaxation(lbm_t* c, double omega_bulk, double omega3, double omega_hi)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    NOT_MID_STEP(c, "lbm_set_relaxation");
    if (!(omega_bulk > 0.0 && omega_bulk < 2.0) || !(omega3 > 0.0 && omega3 < 2.0) || !(omega_hi > 0.0 && omega_hi < 2.0)) {
        set_err("relaxation rates must be in (0,2)");
        return LBM_E_ARG;
    }
    c->omega_bulk = omega_bulk; c->omega3 = omega3; c->omega_hi = omega_hi;
    drop_graph(c);
    return LBM_OK;
}

int lbm_set_trt_magic(lbm_t* c, double lambda)
{
    if (!c || !(lambda > 0.0)) { set_err("magic parameter must be positive"); return LBM_E_ARG; }
    NOT_MID_STEP(c, "lbm_set_trt_magic");
    c->trt_magic = lambda;
    drop_graph(c);
    return LBM_OK;
}

int lbm_init_equilibrium_device(lbm_t* c, const void* rho, const void* u)
{
    if (!c || !rho || !u) { set_err("null argument"); return LBM_E_ARG; }
    const bool ext = !model_is_w2(c->model);
    if (c->dtype == LBM_F64)
        CK(aux_init_equilibrium<double>(c->Q, ext, c->soa, (double*)c->pop[0], c->code, c->g, (const double*)rho,
                                        (const double*)u, c->stream));
    else
        CK(aux_init_equilibrium<float>(c->Q, ext, c->soa, (float*)c->pop[0], c->code, c->g, (const float*)rho,
                                       (const float*)u, c->stream));
    c->launches++;
    c->sto = STO_CANON;
    c->steps = 0;
    c->mid_step = 0;
    c->halo_mode = HALO_NONE;
    return LBM_OK;
}

int lbm_init_equilibrium(lbm_t* c, const void* rho, const void* u)
{
    if (!c || !rho || !u) { set_err("null argument"); return LBM_E_ARG; }
    const size_t nb = (size_t)c->g.n * c->elem;
    char* sc = (char*)scratch_get(c, 4 * nb);
    if (!sc) { set_err("device allocation failed (rho, u staging)"); return LBM_E_ALLOC; }
    CK(cudaMemcpyAsync(sc, rho, nb, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(sc + nb, u, 3 * nb, cudaMemcpyHostToDevice, c->stream));
    if (int rc = lbm_init_equilibrium_device(c, sc, sc + nb)) return rc;
    CK(cudaStreamSynchronize(c->stream));  // host buffers are only read during the call
    scratch_release(c);
    return LBM_OK;
}

int lbm_step(lbm_t* c, int n)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (n < 0) { set_err("n must be >= 0"); return LBM_E_ARG; }
    if (c->sto == STO_NONE) { set_err("lbm_step before lbm_init_equilibrium / lbm_set_populations"); return LBM_E_STATE; }
    if (c->mid_step) { set_err("lbm_step between lbm_step_begin and lbm_step_finish"); return LBM_E_STATE; }
    if (c->has_ghost && n > 0 && (n > 1 || c->fam == FAM_SWAP)) {
        set_err("a context with GHOST cells needs its halo exchanged every step (swap: between the two passes): use lbm_slab_step, or lbm_step_begin ... lbm_step_finish");
        return LBM_E_STATE;
    }
    int s = 0;
    if (graph_wanted(c, n)) {
        // the graph covers an even number of steps from a periodic state: get there first
        if (c->fam == FAM_2POP && use_pull(c) && c->sto == STO_CANON && n > GRAPH_STEPS) {
            if (int rc = one_step(c)) return rc;
            ++s;
        }
        for (; n - s >= GRAPH_STEPS; s += GRAPH_STEPS) {
            int rc = step_graphed(c);
            if (rc == LBM_E_STATE) break;       // capture not possible here: fall back to plain launches
            if (rc != LBM_OK) return rc;
        }
    }
    for (; s < n; ++s)
        if (int rc = one_step(c)) return rc;
    return LBM_OK;
}

int lbm_set_graph(lbm_t* c, int mode)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (mode != LBM_GRAPH_AUTO && mode != LBM_GRAPH_OFF && mode != LBM_GRAPH_ON) { set_err("unknown graph mode %d", mode); return LBM_E_ARG; }
    c->graph_mode = mode;
    drop_graph(c);
    return LBM_OK;
}
long long lbm_graph_replays(const lbm_t* c) { return c ? c->graph_replays : -1; }

int lbm_macroscopic_device(lbm_t* c, void* rho, void* u)
{
    if (!c || !rho || !u) { set_err("null argument"); return LBM_E_ARG; }
    if (c->mid_step) { set_err("export between lbm_step_begin and lbm_step_finish"); return LBM_E_STATE; }
    if (c->sto == STO_NONE) { set_err("no populations loaded"); return LBM_E_STATE; }
    if (c->dtype == LBM_F64)
        CK(aux_macroscopic<double>(c->Q, c->soa, load_mode(c), make_args<double>(c, c->pop[0], nullptr, load_mode(c)), (double*)rho,
                                   (double*)u, c->stream));
    else
        CK(aux_macroscopic<float>(c->Q, c->soa, load_mode(c), make_args<float>(c, c->pop[0], nullptr, load_mode(c)), (float*)rho,
                                  (float*)u, c->stream));
    c->launches++;
    return LBM_OK;
}

int lbm_macroscopic(lbm_t* c, void* rho, void* u)
{
    if (!c || !rho || !u) { set_err("null argument"); return LBM_E_ARG; }
    const size_t nb = (size_t)c->g.n * c->elem;
    char* sc = (char*)scratch_get(c, 4 * nb);
    if (!sc) { set_err("device allocation failed (rho, u staging)"); return LBM_E_ALLOC; }
    if (int rc = lbm_macroscopic_device(c, sc, sc + nb)) return rc;
    CK(cudaMemcpyAsync(rho, sc, nb, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaMemcpyAsync(u, sc + nb, 3 * nb, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    scratch_release(c);
    return LBM_OK;
}

int lbm_kinetic_energy_device(lbm_t* c, double* e_dev)
{
    if (!c || !e_dev) { set_err("null argument"); return LBM_E_ARG; }
    if (c->mid_step) { set_err("export between lbm_step_begin and lbm_step_finish"); return LBM_E_STATE; }
    if (c->sto == STO_NONE) { set_err("no populations loaded"); return LBM_E_STATE; }
    if (c->dtype == LBM_F64)
        CK(aux_energy<double>(c->Q, c->soa, load_mode(c), make_args<double>(c, c->pop[0], nullptr, load_mode(c)), c->partial,
                              c->n_partial, e_dev, c->stream));
    else
        CK(aux_energy<float>(c->Q, c->soa, load_mode(c), make_args<float>(c, c->pop[0], nullptr, load_mode(c)), c->partial,
                             c->n_partial, e_dev, c->stream));
    c->launches += 3;
    return LBM_OK;
}

int lbm_kinetic_energy(lbm_t* c, double* e)
{
    if (!c || !e) { set_err("null argument"); return LBM_E_ARG; }
    if (int rc = lbm_kinetic_energy_device(c, c->e_dev)) return rc;
    CK(cudaMemcpyAsync(e, c->e_dev, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return LBM_OK;
}

// canonical planes f_k of the whole box (cells_dev == nullptr, m = N) or of m listed cells
static int export_planes(lbm_t* c, void* f, const int* cells_dev, int m)
{
    if (c->mid_step) { set_err("export between lbm_step_begin and lbm_step_finish"); return LBM_E_STATE; }
    const size_t nb = (size_t)m * c->elem;
    const size_t plane = ((size_t)m * c->elem + 255) / 256 * 256;
    const int mode = load_mode(c);
    char* sc = (char*)scratch_get(c, 4 * plane);
    if (!sc) { set_err("device allocation failed (plane staging)"); return LBM_E_ALLOC; }
    // scratch planes alternate so that the copy of plane k overlaps nothing it still needs
    for (int k = 0; k < c->Q; ++k) {
        const int kb = c->opp[k];
        PlaneArgs p;
        p.weight = c->w[k];
        const double cu = c->c[kb][0] * c->u_wall[0] + c->c[kb][1] * c->u_wall[1] + c->c[kb][2] * c->u_wall[2];
        p.wterm = -6.0 * c->w[kb] * cu;
        if (mode == LD_LOCAL) { p.slot_fluid = c->sslot[k]; p.slot_wall = c->sslot[k]; p.sx = p.sy = p.sz = 0; }
        else {
            p.slot_fluid = c->sslot[mode == LD_PULL ? k : kb];
            p.slot_wall = c->sslot[mode == LD_PULL ? kb : k];
            p.sx = c->c[k][0]; p.sy = c->c[k][1]; p.sz = c->c[k][2];
        }
        char* out = sc + (size_t)(k & 3) * plane;
        if (c->dtype == LBM_F64)
            CK(aux_extract_plane<double>(c->Q, c->soa, (const double*)c->pop[0], c->code, c->g, p, (double*)out, cells_dev, m, c->stream));
        else
            CK(aux_extract_plane<float>(c->Q, c->soa, (const float*)c->pop[0], c->code, c->g, p, (float*)out, cells_dev, m, c->stream));
        c->launches++;
        CK(cudaMemcpyAsync((char*)f + (size_t)k * nb, out, nb, cudaMemcpyDeviceToHost, c->stream));
    }
    CK(cudaStreamSynchronize(c->stream));
    scratch_release(c);
    return LBM_OK;
}

int lbm_get_populations(lbm_t* c, void* f)
{
    if (!c || !f) { set_err("null argument"); return LBM_E_ARG; }
    if (c->sto == STO_NONE) { set_err("no populations loaded"); return LBM_E_STATE; }
    return export_planes(c, f, nullptr, c->g.n);
}

int lbm_get_populations_at(lbm_t* c, const int32_t* cells, int m, void* f)
{
    if (!c || !f || (!cells && m > 0)) { set_err("null argument"); return LBM_E_ARG; }
    if (m < 0 || m > c->g.n) { set_err("m must be in [0, N]"); return LBM_E_ARG; }
    if (c->sto == STO_NONE) { set_err("no populations loaded"); return LBM_E_STATE; }
    if (m == 0) return LBM_OK;
    for (int t = 0; t < m; ++t)
        if (cells[t] < 0 || cells[t] >= c->g.n) { set_err("cell index %d out of range at position %d", cells[t], t); return LBM_E_ARG; }
    int* cells_dev = (int*)dev_alloc(c, sizeof(int) * (size_t)m);
    if (!cells_dev) { set_err("device allocation failed"); return LBM_E_ALLOC; }
    c->dev_bytes -= (long long)(sizeof(int) * (size_t)m);  // transient
    int rc = LBM_OK;
    if (cudaMemcpyAsync(cells_dev, cells, sizeof(int) * (size_t)m, cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        rc = cuda_fail("cell list upload", cudaGetLastError());
    if (rc == LBM_OK) rc = export_planes(c, f, cells_dev, m);
    cudaStreamSynchronize(c->stream);
    dev_free(c, cells_dev);
    return rc;
}

int lbm_set_populations(lbm_t* c, const void* f)
{
    if (!c || !f) { set_err("null argument"); return LBM_E_ARG; }
    const size_t nb = (size_t)c->g.n * c->elem;
    char* sc = (char*)scratch_get(c, 4 * nb);
    if (!sc) { set_err("device allocation failed (plane staging)"); return LBM_E_ALLOC; }
    drop_graph(c);
    for (int k = 0; k < c->Q; ++k) {
        char* in = sc + (size_t)(k & 3) * nb;
        CK(cudaMemcpyAsync(in, (const char*)f + (size_t)k * nb, nb, cudaMemcpyHostToDevice, c->stream));
        if (c->dtype == LBM_F64)
            CK(aux_insert_plane<double>(c->Q, c->soa, (double*)c->pop[0], c->code, c->g, c->sslot[k], c->w[k], (const double*)in, c->stream));
        else
            CK(aux_insert_plane<float>(c->Q, c->soa, (float*)c->pop[0], c->code, c->g, c->sslot[k], c->w[k], (const float*)in, c->stream));
        c->launches++;
    }
    CK(cudaStreamSynchronize(c->stream));
    scratch_release(c);
    c->sto = STO_CANON;
    c->mid_step = 0;
    c->halo_mode = HALO_NONE;
    return LBM_OK;
}

// ---- slab decomposition along x: the time step in parts, halo pack / unpack, and the
// driver that pushes the boundary populations straight into the neighbouring slab's receive buffer
static int slab_check(lbm_t* c, const char* what)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (!c->soa || (c->fam == FAM_2POP && !use_pull(c))) {
        set_err("%s: the slab calls exist for the SoA schemes (two-population pull form, swap, AA) only", what);
        return LBM_E_ARG;
    }
    if (c->sto == STO_NONE) { set_err("%s before lbm_init_equilibrium / lbm_set_populations", what); return LBM_E_STATE; }
    return LBM_OK;
}
// which step kernel the next step of the context's scheme runs on its cells (Table 1)
static int next_kind(const lbm_t* c)
{
    if (c->fam == FAM_2POP) return c->sto == STO_CANON ? SK_COLLIDE : SK_PULL;
    if (c->fam == FAM_AA) return c->sto == STO_CANON ? SK_EVEN : SK_ODD;
    return SK_EVEN;   // swap pass 1
}
// one launch of that kernel over the x-layers [xa, xb), nothing committed
static int step_layers(lbm_t* c, int xa, int xb)
{
    if (xb <= xa) return LBM_OK;
    const int layer = c->ny * c->nz;
    c->range_first = xa * layer;
    c->range_end = xb * layer;
    const int kind = next_kind(c);
    cudaError_t e = step_kind(c, kind, c->pop[0], kind == SK_PULL ? c->pop[1] : c->pop[0]);
    c->range_first = c->range_end = 0;
    if (e != cudaSuccess) return cuda_fail("step_layers", e);
    return LBM_OK;
}
int lbm_step_begin(lbm_t* c)
{
    if (int rc = slab_check(c, "lbm_step_begin")) return rc;
    if (c->mid_step) { set_err("lbm_step_begin twice"); return LBM_E_STATE; }
    if (c->outer_fluid) {
        set_err("lbm_step_begin: the x-layers 0 and nx-1 are not updated by the split step and must hold no FLUID cell (GHOST or solid)");
        return LBM_E_STATE;
    }
    const int kind = next_kind(c);
    if (int rc = step_layers(c, 1, 2)) return rc;
    if (c->nx - 2 > 1)
        if (int rc = step_layers(c, c->nx - 2, c->nx - 1)) return rc;
    c->halo_mode = kind == SK_ODD ? HALO_PUSHED : c->fam == FAM_2POP ? HALO_POST_K : HALO_POST_KBAR;
    c->mid_step = 1;
    return LBM_OK;
}
int lbm_step_end(lbm_t* c)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (c->mid_step != 1) { set_err("lbm_step_end without lbm_step_begin"); return LBM_E_STATE; }
    if (int rc = step_layers(c, 2, c->nx - 2)) return rc;
    if (c->fam == FAM_2POP) {
        if (c->sto == STO_CANON) c->sto = STO_POST;
        else { void* t = c->pop[0]; c->pop[0] = c->pop[1]; c->pop[1] = t; }
    } else if (c->fam == FAM_AA) {
        c->sto = c->sto == STO_CANON ? STO_AA_ODD : STO_CANON;
    }
    c->mid_step = 2;
    return LBM_OK;
}
int lbm_step_finish(lbm_t* c)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (c->mid_step != 2) { set_err("lbm_step_finish without lbm_step_end"); return LBM_E_STATE; }
    if (c->fam == FAM_SWAP)
        if (int rc = swap_pass2(c)) return rc;
    c->mid_step = 0;
    c->steps++;
    return LBM_OK;
}

long long lbm_halo_count(const lbm_t* c)
{
    if (!c) return -1;
    return (long long)(c->Q == 19 ? 5 : 9) * c->ny * c->nz;
}
// the directions with c_x = want_cx, in increasing k
static void halo_dirs(const lbm_t* c, int want_cx, HaloArgs* p, bool opposite_slot)
{
    p->ndir = 0;
    for (int k = 0; k < c->Q; ++k)
        if (c->c[k][0] == want_cx) {
            p->slot[p->ndir] = opposite_slot ? c->opp[k] : k;
            p->cy[p->ndir] = c->c[k][1];
            p->cz[p->ndir] = c->c[k][2];
            p->ndir++;
        }
    p->ny = c->ny; p->nz = c->nz;
    p->cells = c->ny * c->nz;
    p->merge = 0;
    p->first = p->up_first = 0;
    p->flag = nullptr; p->seq = 0; p->counter = nullptr; p->status = nullptr;
}
static int halo_launch(lbm_t* c, bool pack, void* pop, const HaloArgs& p, void* buf)
{
    if (c->dtype == LBM_F64) CK(aux_halo<double>(pack, (double*)pop, c->code, c->g.stride, p, (double*)buf, c->stream));
    else CK(aux_halo<float>(pack, (float*)pop, c->code, c->g.stride, p, (float*)buf, c->stream));
    c->launches++;
    return LBM_OK;
}
// what leaves through `face` (0: low x, 1: high x) after the step part that ran last
static int halo_pack_args(lbm_t* c, int face, HaloArgs* p, void** from)
{
    if (c->halo_mode == HALO_NONE) { set_err("lbm_halo_pack: no step has run since the populations were loaded"); return LBM_E_STATE; }
    const long long layer = (long long)c->ny * c->nz;
    const int cx = face == 0 ? -1 : +1;
    *from = c->pop[0];
    if (c->halo_mode == HALO_PUSHED) {
        // AA odd step: the outermost owned layer has pushed into the ghost layer (slot k of x + c_k)
        halo_dirs(c, cx, p, false);
        p->first = (face == 0 ? 0 : c->nx - 1) * layer;
    } else {
        // post-collision values of the outermost owned layer: slot k (two-population) or kbar (AA even, swap pass 1)
        halo_dirs(c, cx, p, c->halo_mode == HALO_POST_KBAR);
        p->first = (face == 0 ? 1 : c->nx - 2) * layer;
        // two-population: between lbm_step_begin and lbm_step_end the new values sit in the array being written
        if (c->fam == FAM_2POP && c->mid_step == 1 && c->sto == STO_POST) *from = c->pop[1];
    }
    return LBM_OK;
}
// where what entered through `face` goes
static int halo_unpack_args(lbm_t* c, int face, HaloArgs* p)
{
    if (c->halo_mode == HALO_NONE) { set_err("lbm_halo_unpack: no step has run since the populations were loaded"); return LBM_E_STATE; }
    if (c->mid_step == 1) { set_err("lbm_halo_unpack between lbm_step_begin and lbm_step_end"); return LBM_E_STATE; }
    if (c->fam == FAM_SWAP && c->mid_step != 2) { set_err("swap scheme: lbm_halo_unpack belongs between lbm_step_end and lbm_step_finish (pass 2 needs the halo)"); return LBM_E_STATE; }
    const long long layer = (long long)c->ny * c->nz;
    const int cx = face == 0 ? +1 : -1;   // what enters through the low face moves towards +x
    const long long ghost = (face == 0 ? 0 : c->nx - 1) * layer, owned = (face == 0 ? 1 : c->nx - 2) * layer;
    if (c->halo_mode == HALO_PUSHED) {
        halo_dirs(c, cx, p, false);
        p->first = owned; p->up_first = ghost; p->merge = 1;
    } else if (c->fam == FAM_SWAP && face == 1) {
        // pass 2 exchanges pop_kbar(y) <-> pop_k(y + c_k) from the cell y with c_k,x = -1; for a ghost y
        // that thread does not exist here, so its half of the exchange is done on arrival:
        // pop_k(x) <- f_out_k(y) = the neighbour's pop_kbar(y), x = y + c_k in the last owned layer
        halo_dirs(c, cx, p, false);
        p->first = owned; p->up_first = ghost; p->merge = 2;
    } else {
        halo_dirs(c, cx, p, c->halo_mode == HALO_POST_KBAR);
        p->first = ghost;
    }
    return LBM_OK;
}
static int halo_face_check(lbm_t* c, int face, const void* buf, const char* what)
{
    if (int rc = slab_check(c, what)) return rc;
    if (!buf) { set_err("null argument"); return LBM_E_ARG; }
    if (face != 0 && face != 1) { set_err("face must be 0 (low x) or 1 (high x)"); return LBM_E_ARG; }
    return LBM_OK;
}
int lbm_halo_pack(lbm_t* c, int face, void* buf)
{
    if (int rc = halo_face_check(c, face, buf, "lbm_halo_pack")) return rc;
    HaloArgs p; void* from;
    if (int rc = halo_pack_args(c, face, &p, &from)) return rc;
    return halo_launch(c, true, from, p, buf);
}
int lbm_halo_unpack(lbm_t* c, int face, const void* buf)
{
    if (int rc = halo_face_check(c, face, buf, "lbm_halo_unpack")) return rc;
    HaloArgs p;
    if (int rc = halo_unpack_args(c, face, &p)) return rc;
    return halo_launch(c, false, c->pop[0], p, const_cast<void*>(buf));
}

// the slab driver may be called for contexts on several devices from one host thread (one process, peer
// access): it makes the context's device current for the duration of the call
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// ---- the driver: boundary layers -> peer store -> interior -> merge, without the host in between
// One allocation per context (cudaMalloc, so that it can be shared through CUDA IPC):
//   recv[face][parity][halo_count] elements | flag[face] (u64) | counter[face] (u32) | status (int)
static size_t slab_buf_bytes(const lbm_t* c) { return ((size_t)lbm_halo_count(c) * c->elem + 255) / 256 * 256; }
static char* slab_recv(const lbm_t* c, char* base, int face, int parity) { return base + (size_t)(face * 2 + parity) * slab_buf_bytes(c); }
static char* slab_tail(const lbm_t* c, char* base) { return base + 4 * slab_buf_bytes(c); }
static unsigned long long* slab_flag(const lbm_t* c, char* base, int face) { return reinterpret_cast<unsigned long long*>(slab_tail(c, base)) + face; }
static unsigned* slab_counter(const lbm_t* c, char* base, int face) { return reinterpret_cast<unsigned*>(slab_tail(c, base) + 16) + face; }
static int* slab_status(const lbm_t* c, char* base) { return reinterpret_cast<int*>(slab_tail(c, base) + 24); }
static int slab_alloc(lbm_t* c)
{
    if (c->slab_mem) return LBM_OK;
    const size_t bytes = 4 * slab_buf_bytes(c) + 64;
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); set_err("device allocation failed (halo receive buffers)"); return LBM_E_ALLOC; }
    CK(cudaMemsetAsync(p, 0, bytes, c->stream));
    c->slab_mem = (char*)p;
    c->dev_bytes += (long long)bytes;
    return LBM_OK;
}
int lbm_slab_link(lbm_t* c, int face, lbm_t* peer)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (!c->soa) { set_err("lbm_slab_link: SoA schemes only"); return LBM_E_ARG; }
    if (face != 0 && face != 1) { set_err("face must be 0 (low x) or 1 (high x)"); return LBM_E_ARG; }
    if (!peer) { c->peer_mem[face] = nullptr; return LBM_OK; }
    if (peer->ny != c->ny || peer->nz != c->nz || peer->Q != c->Q || peer->dtype != c->dtype || peer->scheme != c->scheme) {
        set_err("lbm_slab_link: the neighbouring slab must have the same ny, nz, lattice, scheme and dtype");
        return LBM_E_ARG;
    }
    if (peer->device != c->device) {   // another GPU of this process: the pack kernel stores into its memory
        int can = 0;
        if (cudaDeviceCanAccessPeer(&can, c->device, peer->device) != cudaSuccess || !can) {
            cudaGetLastError();
            set_err("lbm_slab_link: device %d cannot access the memory of device %d", c->device, peer->device);
            return LBM_E_ARG;
        }
        DeviceGuard g(c->device);
        const cudaError_t e = cudaDeviceEnablePeerAccess(peer->device, 0);
        if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return cuda_fail("cudaDeviceEnablePeerAccess", e);
        cudaGetLastError();
    }
    { DeviceGuard g(c->device); if (int rc = slab_alloc(c)) return rc; }
    { DeviceGuard g(peer->device); if (int rc = slab_alloc(peer)) return rc; }
    c->peer_mem[face] = peer->slab_mem;
    return LBM_OK;
}
int lbm_slab_export(lbm_t* c, void* handle64)
{
    if (!c || !handle64) { set_err("null argument"); return LBM_E_ARG; }
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
    if (int rc = slab_alloc(c)) return rc;
    cudaIpcMemHandle_t h;
    CK(cudaIpcGetMemHandle(&h, c->slab_mem));
    memcpy(handle64, &h, sizeof h);
    return LBM_OK;
}
int lbm_slab_import(lbm_t* c, int face, const void* handle64)
{
    if (!c || !handle64) { set_err("null argument"); return LBM_E_ARG; }
    if (face != 0 && face != 1) { set_err("face must be 0 (low x) or 1 (high x)"); return LBM_E_ARG; }
    if (int rc = slab_alloc(c)) return rc;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle64, sizeof h);
    void* p = nullptr;
    CK(cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess));
    c->peer_mem[face] = (char*)p;
    c->peer_ipc[face] = true;
    return LBM_OK;
}
// first half of a slab step: outermost owned layers, their halo stored into the neighbours' receive
// buffers (sequence number published last), then the interior
int lbm_slab_post(lbm_t* c)
{
    if (int rc = slab_check(c, "lbm_slab_post")) return rc;
    DeviceGuard guard(c->device);
    if (int rc = lbm_step_begin(c)) return rc;
    for (int face = 0; face < 2; ++face) {
        if (!c->peer_mem[face]) continue;
        HaloArgs p; void* from;
        if (int rc = halo_pack_args(c, face, &p, &from)) return rc;
        const unsigned long long seq = ++c->seq_out[face];
        // what leaves through my low face enters the neighbour through its high face
        p.flag = slab_flag(c, c->peer_mem[face], 1 - face);
        p.seq = seq;
        p.counter = slab_counter(c, c->slab_mem, face);
        if (int rc = halo_launch(c, true, from, p, slab_recv(c, c->peer_mem[face], 1 - face, (int)(seq & 1)))) return rc;
    }
    return lbm_step_end(c);
}
// second half: wait for the neighbours' messages, merge them, finish the step (swap: pass 2)
int lbm_slab_complete(lbm_t* c)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (c->mid_step != 2) { set_err("lbm_slab_complete without lbm_slab_post"); return LBM_E_STATE; }
    DeviceGuard guard(c->device);
    for (int face = 0; face < 2; ++face) {
        if (!c->peer_mem[face]) continue;
        HaloArgs p;
        if (int rc = halo_unpack_args(c, face, &p)) return rc;
        const unsigned long long seq = ++c->seq_in[face];
        p.flag = slab_flag(c, c->slab_mem, face);
        p.seq = seq;
        p.status = slab_status(c, c->slab_mem);
        if (int rc = halo_launch(c, false, c->pop[0], p, slab_recv(c, c->slab_mem, face, (int)(seq & 1)))) return rc;
    }
    return lbm_step_finish(c);
}
int lbm_slab_step(lbm_t* c, int n)
{
    if (n < 0) { set_err("n must be >= 0"); return LBM_E_ARG; }
    for (int s = 0; s < n; ++s) {
        if (int rc = lbm_slab_post(c)) return rc;
        if (int rc = lbm_slab_complete(c)) return rc;
    }
    return LBM_OK;
}
int lbm_slab_status(lbm_t* c)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (!c->slab_mem) return LBM_OK;
    int st = 0;
    CK(cudaMemcpyAsync(&st, slab_status(c, c->slab_mem), sizeof st, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (st) { set_err("a halo message did not arrive (the neighbouring slab stopped stepping?)"); return LBM_E_STATE; }
    return LBM_OK;
}

// ---- kinetic energy with its scratch in a fixed device array: an entry point that allocates nothing.
// The reduce kernel (energy_kernel, kernels.cuh) writes one partial sum per block of 256 cells, and two
// summing stages fold them (aux_energy).  lbm_kinetic_energy_device keeps those partials in a buffer that
// lbm_create allocated; here they live in a file-scope array that every GPU which loads the library holds
// until the process exits.  Nothing in the array has to start at zero: every element a call reads it has
// written itself (ceil(N/256) partials, then at most ENERGY_STAGE2 sums), so the contents the last call
// left behind -- of this or of any other context -- are never looked at.
static __device__ __align__(256) double g_static_scratch[LBM_STATIC_SCRATCH_DOUBLES];

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the address the kernels
// need comes from cudaGetSymbolAddress, asked once per device with that device current.
enum { STATIC_MAX_DEVICES = 64 };
static double* g_static_ptr[STATIC_MAX_DEVICES];   // per device, nullptr = not resolved yet

static int static_scratch_ptr(int device, double** out)
{
    if (device < 0 || device >= STATIC_MAX_DEVICES) { set_err("device %d outside [0, %d)", device, (int)STATIC_MAX_DEVICES); return LBM_E_ARG; }
    if (!g_static_ptr[device]) {
        DeviceGuard guard(device);
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess || !p) return cuda_fail("cudaGetSymbolAddress(static scratch)", e);
        g_static_ptr[device] = p;
    }
    *out = g_static_ptr[device];
    return LBM_OK;
}

int lbm_kinetic_energy_device_static(lbm_t* c, double* e_dev)
{
    if (!c || !e_dev) { set_err("null argument"); return LBM_E_ARG; }
    // the partials of this lattice and the sums of the second stage must fit the fixed array
    if ((long long)c->n_partial + ENERGY_STAGE2 > (long long)LBM_STATIC_SCRATCH_DOUBLES) {
        set_err("lbm_kinetic_energy_device_static: %d cells need %d partial sums, the static scratch holds %d doubles "
                "(at most %lld cells); use lbm_kinetic_energy_device", c->g.n, c->n_partial + (int)ENERGY_STAGE2,
                (int)LBM_STATIC_SCRATCH_DOUBLES, (long long)LBM_STATIC_MAX_CELLS);
        return LBM_E_ARG;
    }
    if (c->mid_step) { set_err("export between lbm_step_begin and lbm_step_finish"); return LBM_E_STATE; }
    if (c->sto == STO_NONE) { set_err("no populations loaded"); return LBM_E_STATE; }
    double* scratch = nullptr;
    if (int rc = static_scratch_ptr(c->device, &scratch)) return rc;
    if (c->dtype == LBM_F64)
        CK(aux_energy<double>(c->Q, c->soa, load_mode(c), make_args<double>(c, c->pop[0], nullptr, load_mode(c)), scratch,
                              c->n_partial, e_dev, c->stream));
    else
        CK(aux_energy<float>(c->Q, c->soa, load_mode(c), make_args<float>(c, c->pop[0], nullptr, load_mode(c)), scratch,
                             c->n_partial, e_dev, c->stream));
    c->launches += 3;
    return LBM_OK;
}

long long lbm_steps_done(const lbm_t* c) { return c ? c->steps : -1; }
long long lbm_num_fluid(const lbm_t* c) { return c ? c->n_fluid : -1; }
long long lbm_device_bytes(const lbm_t* c) { return c ? c->dev_bytes : -1; }
long long lbm_kernel_launches(const lbm_t* c) { return c ? c->launches : -1; }

int lbm_sync(lbm_t* c)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    CK(cudaStreamSynchronize(c->stream));
    return LBM_OK;
}

int lbm_set_block(lbm_t* c, int threads)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (threads < 32 || threads > 256 || (threads & 31)) { set_err("threads per block must be a multiple of 32 in [32, 256]"); return LBM_E_ARG; }
    NOT_MID_STEP(c, "lbm_set_block");
    c->block = threads;
    drop_graph(c);
    return LBM_OK;
}

int lbm_set_variant(lbm_t* c, int variant)
{
    if (!c) { set_err("null context"); return LBM_E_ARG; }
    if (variant < 0 || variant >= V_COUNT) { set_err("unknown variant %d", variant); return LBM_E_ARG; }
    NOT_MID_STEP(c, "lbm_set_variant");
    if (variant == V_GENERIC_PUSH && c->has_ghost) { set_err("the generic_push variant has no halo exchange: not with LBM_GHOST cells"); return LBM_E_ARG; }
    if (c->fam == FAM_2POP && variant == V_GENERIC_PUSH) {
        if (int rc = normalise(c)) return rc;
    }
    c->variant = variant;
    c->pdl = variant != V_PLAIN;
    c->prefetch = variant == V_PLAIN ? 0 : -1;
    drop_graph(c);
    return LBM_OK;
}

}  // extern "C"
