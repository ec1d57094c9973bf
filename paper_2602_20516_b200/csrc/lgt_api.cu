// lgt_api.cu -- the C ABI of include/lgt.h: handle, argument checks, kernel launches.
// No torch, no host-side arithmetic on fields: every step of the path runs in the kernels of kernels.cuh.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

#include "../../include/lgt.h"
#include "kernels.cuh"

using namespace lgt;

namespace {
std::string g_create_error;
}

constexpr int LGT_MAX_SMEAR = 8;

struct lgt_ctx {
    Geom g;
    double beta, kappa;
    int prec;
    int device;
    cudaStream_t stream;
    size_t esize;  // bytes of one complex number
    void* U = nullptr;    // native links   [36][Vs] complex
    void* P = nullptr;    // native momenta [16][Vs] pairs
    void* phi = nullptr;  // native pseudofermion
    bool has_phi = false;
    void* ws[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // x, r, p, t, (spare), b
    // mixed-precision solver (LGT_F64 handles only, lazy): fp32 copy of the links, five fp32 spinor workspaces
    void* U32 = nullptr;
    bool u32_valid = false;
    void* ws32[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};  // b, e, r, p, t
    // even/odd preconditioned action (lazy): checkerboard copy of the links, eight half spinor fields
    int action = LGT_ACTION_FULL;
    void* Ucb = nullptr;
    bool ucb_valid = false;
    void* eo = nullptr;  // Xe, Xo, Ye, Yo, be, re, pe, to: 8 x 12 * Vhs complex
    // mixed-precision solve of the even/odd system (LGT_F64 handles, lazy): fp32 checkerboard links, six fp32 half fields
    void* Ucb32 = nullptr;
    bool ucb32_valid = false;
    void* eo32 = nullptr;  // b, e, r, p, u, t
    int solver = LGT_SOLVER_CG;
    // stout smearing of the links the fermions see (lazy): Usm[k] = level k+1 links, Asm[k] = its exponents (compact)
    int nsmear = 0;
    double rho = 0.0;
    void* Usm[LGT_MAX_SMEAR] = {};
    void* Asm[LGT_MAX_SMEAR] = {};
    bool usm_valid = false;
    void* Uf = nullptr;  // links of the Dirac operator: U, or Usm[nsmear - 1]
    void* F2 = nullptr;  // three more compact force buffers for the smearing recursion (lazy)
    void* F3 = nullptr;
    void* F4 = nullptr;
    // a time slab of a decomposed lattice (lgt_dd_*): the group's "link ghosts are current" flag, cleared on link changes
    bool* dd_links_valid = nullptr;
    int integrator = LGT_INT_LEAPFROG;
    int n_inner = 1;        // gauge sub-steps per step of the Sexton-Weingarten integrator
    void* Usave = nullptr;  // links at the start of an HMC trajectory (lazy)
    double inner_tol = 1e-5;
    int last_outer = 0;
    void* F = nullptr;      // compact force buffer for the canonical-output calls (lazy)
    void* stage = nullptr;  // canonical staging buffer for *_host calls and conversions (lazy)
    // asynchronous host transfers (lgt_*_host_async): a copy stream, a staging buffer per transfer kind, and the events that
    // order them against the handle's stream (lazy)
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_main = nullptr, ev_p_up = nullptr, ev_u_down = nullptr, ev_p_down = nullptr;
    void* stage_p_in = nullptr;
    void* stage_u_out = nullptr;
    void* stage_p_out = nullptr;
    bool p_pending = false, u_down_pending = false, p_down_pending = false;
    size_t stage_bytes = 0;
    double* partials = nullptr;
    unsigned* counter = nullptr;
    CgState* st = nullptr;
    bool fold_default = false;
    bool inner_exact = false;  // the fp32 inner hops of the mixed even/odd solver stopped contracting on 12-real links: exact links until the links change
    CgState* st2 = nullptr;  // the second state of the folded scalar updates (LGT_K_CG_BLAS variant 3): iterations alternate
    double* scal = nullptr;  // device result slots
    CgState* h_st = nullptr;  // pinned
    double* h_scal = nullptr;  // pinned
    int red_blocks = 0;
    int num_sms = 0;
    int variant[LGT_K_COUNT] = {};  // kernel variant per class (lgt_set_kernel_variant)
    bool coop_default = false;  // set once the one-launch CG has been measured faster (lgt_create)
    unsigned* coop_counter = nullptr;  // grid barrier of the cooperative CG kernels (lazy, zero between launches)
    long launches = 0;
    // optional CUDA-event timing of every launch, by kernel class (lgt_timing_*)
    bool timing = false;
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    std::vector<int> ev_class;  // class of the launch bracketed by events (2i, 2i+1)
    // CUDA graphs of one chunk (8 iterations) of the CG loops, keyed by the buffers the chunk touches (lazy)
    struct ChunkGraph {
        int kind;
        const void* key[7];
        int swz;
        cudaGraphExec_t exec;
        int launches;
    };
    std::vector<ChunkGraph> graphs;
    cudaStream_t capture_stream = nullptr;
    bool graphs_ok = true;
    std::string err;
};

namespace {

int fail(lgt_ctx* c, int code, const char* what, cudaError_t e = cudaSuccess) {
    char buf[512];
    if (e != cudaSuccess)
        snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    else
        snprintf(buf, sizeof buf, "%s", what);
    if (c)
        c->err = buf;
    else
        g_create_error = buf;
    return code;
}

#define CU(call)                                                                  \
    do {                                                                          \
        cudaError_t e_ = (call);                                                  \
        if (e_ != cudaSuccess) return fail(c, (e_ == cudaErrorMemoryAllocation) ? LGT_ENOMEM : LGT_ECUDA, #call, e_); \
    } while (0)

cudaEvent_t timing_event(lgt_ctx* c) {
    if (c->ev_used == c->ev_pool.size()) {
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
        c->ev_pool.push_back(e);
    }
    return c->ev_pool[c->ev_used++];
}

#define LAUNCH(c, kclass, kern, grid, block, ...)                   \
    do {                                                            \
        cudaEvent_t e0_ = nullptr, e1_ = nullptr;                   \
        if ((c)->timing) {                                          \
            e0_ = timing_event(c);                                  \
            e1_ = timing_event(c);                                  \
            if (e0_ && e1_) {                                       \
                (c)->ev_class.push_back(kclass);                    \
                cudaEventRecord(e0_, (c)->stream);                  \
            }                                                       \
        }                                                           \
        kern<<<(grid), (block), 0, (c)->stream>>>(__VA_ARGS__);     \
        if (e0_ && e1_) cudaEventRecord(e1_, (c)->stream);          \
        (c)->launches++;                                            \
        cudaError_t e_ = cudaGetLastError();                        \
        if (e_ != cudaSuccess) return fail((c), LGT_ECUDA, #kern, e_); \
    } while (0)

// the same with dynamic shared memory (opt-in above 48 KB)
#define LAUNCH_SMEM(c, kclass, kern, grid, block, smem, ...)        \
    do {                                                            \
        {   /* per device, so set on every launch (a host-side table lookup) */ \
            cudaError_t ea_ = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (smem)); \
            if (ea_ != cudaSuccess) return fail((c), LGT_ECUDA, "cudaFuncSetAttribute " #kern, ea_); \
        }                                                           \
        cudaEvent_t e0_ = nullptr, e1_ = nullptr;                   \
        if ((c)->timing) {                                          \
            e0_ = timing_event(c);                                  \
            e1_ = timing_event(c);                                  \
            if (e0_ && e1_) {                                       \
                (c)->ev_class.push_back(kclass);                    \
                cudaEventRecord(e0_, (c)->stream);                  \
            }                                                       \
        }                                                           \
        kern<<<(grid), (block), (smem), (c)->stream>>>(__VA_ARGS__); \
        if (e0_ && e1_) cudaEventRecord(e1_, (c)->stream);          \
        (c)->launches++;                                            \
        cudaError_t e_ = cudaGetLastError();                        \
        if (e_ != cudaSuccess) return fail((c), LGT_ECUDA, #kern, e_); \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) {
        cudaGetDevice(&prev);
        if (prev != dev) cudaSetDevice(dev);
        else prev = -1;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

inline size_t spinor_bytes(const lgt_ctx* c) { return (size_t)12 * c->g.Vs * c->esize; }
inline size_t links_bytes(const lgt_ctx* c) { return (size_t)36 * c->g.Vs * c->esize; }
inline size_t mom_bytes(const lgt_ctx* c) { return (size_t)16 * c->g.Vs * c->esize; }
// sites the compute kernels own (Geom::s_begin .. s_end), padding lanes included on an undivided lattice
inline int own_sites(const lgt_ctx* c) { return (c->g.s_end == c->g.V ? c->g.Vs : c->g.s_end) - c->g.s_begin; }
inline int site_blocks(const lgt_ctx* c, int bs) { return (own_sites(c) + bs - 1) / bs; }
// the same for one parity of a checkerboarded field
inline int own_half_sites(const lgt_ctx* c) { return (c->g.h_end == c->g.Vh ? c->g.Vhs : c->g.h_end) - c->g.h_begin; }
inline int stream_blocks(const lgt_ctx* c, size_t n) {
    size_t b = (n + 255) / 256;
    return (int)(b < (size_t)c->red_blocks ? (b ? b : 1) : c->red_blocks);
}

int ensure_stage(lgt_ctx* c, size_t bytes) {
    if (c->stage_bytes >= bytes) return LGT_OK;
    if (c->stage) cudaFree(c->stage);
    c->stage = nullptr;
    c->stage_bytes = 0;
    CU(cudaMalloc(&c->stage, bytes));
    c->stage_bytes = bytes;
    return LGT_OK;
}
int ensure_force_buf(lgt_ctx* c) {
    if (c->F) return LGT_OK;
    CU(cudaMalloc(&c->F, mom_bytes(c)));
    return LGT_OK;
}

// An asynchronous upload of the momenta (lgt_set_momenta_host_async) may still be in flight on the copy stream: whoever is
// about to launch a kernel that touches c->P first makes the handle's stream wait for it.
inline void p_ready(lgt_ctx* c) {
    if (c->p_pending) {
        cudaStreamWaitEvent(c->stream, c->ev_p_up, 0);
        c->p_pending = false;
    }
}

// every copy derived from the links (fp32, checkerboard, smeared, the slabs' ghost slices) is stale after a link change
inline void invalidate_link_copies(lgt_ctx* c) {
    c->u32_valid = false;
    c->usm_valid = false;
    if (c->dd_links_valid) *c->dd_links_valid = false;
    c->ucb_valid = false;
    c->ucb32_valid = false;
    c->inner_exact = false;
}

int eo_cg_mixed(lgt_ctx* c, void* b, void* x, void* r, void* q, void* u, void* t_o, double tol, int max_iter, int* iters);

// One chunk of CG iterations as a CUDA graph: the kernels of a chunk have no argument that changes from chunk to chunk
// (the scalars, the stop flag and the "update due" flag live on the device), so the first chunk on a given set of buffers
// is captured -- on a side stream, since the handle's stream may be the legacy default stream, which cannot capture --
// and every later one is a single cudaGraphLaunch on the handle's stream.  This takes the per-launch host cost out of
// the loop, which is what bounds small lattices (16^4: 7 launches of 3-10 us of work each per iteration).  Falls back to
// plain launches while per-kernel timing is on, or if capture is not possible.
template <class Body> int chunk_graph(lgt_ctx* c, int kind, const void* const (&key)[7], Body body) {
    if (c->timing || !c->graphs_ok) return body();
    for (const lgt_ctx::ChunkGraph& g : c->graphs)
        if (g.kind == kind && g.swz == c->g.swz_Z && memcmp(g.key, key, sizeof key) == 0) {
            CU(cudaGraphLaunch(g.exec, c->stream));
            c->launches += g.launches;
            return LGT_OK;
        }
    if (!c->capture_stream && cudaStreamCreateWithFlags(&c->capture_stream, cudaStreamNonBlocking) != cudaSuccess) {
        c->graphs_ok = false;
        cudaGetLastError();
        return body();
    }
    cudaStream_t user = c->stream;
    const long l0 = c->launches;
    if (cudaStreamBeginCapture(c->capture_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        c->graphs_ok = false;
        cudaGetLastError();
        return body();
    }
    c->stream = c->capture_stream;
    const int rc = body();
    c->stream = user;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->capture_stream, &graph);
    const int nl = (int)(c->launches - l0);
    c->launches = l0;
    cudaGraphExec_t exec = nullptr;
    if (rc == LGT_OK && e == cudaSuccess && graph) e = cudaGraphInstantiate(&exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (rc != LGT_OK || e != cudaSuccess || !exec) {
        c->graphs_ok = false;
        cudaGetLastError();
        return body();
    }
    lgt_ctx::ChunkGraph g;
    g.kind = kind;
    memcpy(g.key, key, sizeof key);
    g.swz = c->g.swz_Z;
    g.exec = exec;
    g.launches = nl;
    if (c->graphs.size() >= 16) {  // buffers keep changing (caller-owned x): do not hoard
        cudaGraphExecDestroy(c->graphs.front().exec);
        c->graphs.erase(c->graphs.begin());
    }
    c->graphs.push_back(g);
    CU(cudaGraphLaunch(exec, c->stream));
    c->launches += nl;
    return LGT_OK;
}

template <class T> struct Ops {
    typedef typename Vec2<T>::type T2;

    static int to_native(lgt_ctx* c, const void* src, void* dst, int ncomp) {
        size_t n = (size_t)c->g.Vs * ncomp;
        if (ncomp == 36)
            LAUNCH(c, LGT_K_OTHER, (reorder_kernel<T, 0, 36, 1>), stream_blocks(c, n), 256, c->g, (const T2*)src, (T2*)dst);
        else
            LAUNCH(c, LGT_K_OTHER, (reorder_kernel<T, 0, 12, 0>), stream_blocks(c, n), 256, c->g, (const T2*)src, (T2*)dst);
        return LGT_OK;
    }
    static int from_native(lgt_ctx* c, const void* src, void* dst, int ncomp) {
        size_t n = (size_t)c->g.Vs * ncomp;
        if (ncomp == 36)
            LAUNCH(c, LGT_K_OTHER, (reorder_kernel<T, 1, 36, 1>), stream_blocks(c, n), 256, c->g, (const T2*)src, (T2*)dst);
        else
            LAUNCH(c, LGT_K_OTHER, (reorder_kernel<T, 1, 12, 0>), stream_blocks(c, n), 256, c->g, (const T2*)src, (T2*)dst);
        return LGT_OK;
    }
    static int momenta_to_native(lgt_ctx* c, const void* src, void* dst) {
        LAUNCH(c, LGT_K_OTHER, (momenta_reorder_kernel<T, 0>), stream_blocks(c, (size_t)4 * c->g.Vs), 256, c->g, (const T2*)src, (T2*)dst);
        return LGT_OK;
    }
    static int momenta_from_native(lgt_ctx* c, const void* src, void* dst) {
        LAUNCH(c, LGT_K_OTHER, (momenta_reorder_kernel<T, 1>), stream_blocks(c, (size_t)4 * c->g.Vs), 256, c->g, (const T2*)src, (T2*)dst);
        return LGT_OK;
    }
    static int unit_links(lgt_ctx* c) {
        c->u32_valid = false;
    c->usm_valid = false;
    if (c->dd_links_valid) *c->dd_links_valid = false;
        c->ucb_valid = false;
    c->ucb32_valid = false;
    c->inner_exact = false;
        LAUNCH(c, LGT_K_OTHER, (unit_links_kernel<T>), stream_blocks(c, (size_t)36 * c->g.Vs), 256, c->g, (T2*)c->U);
        return LGT_OK;
    }

    // dslash_tile_kernel's preconditions (an undivided lattice whose xy planes split into 64-site runs, even Lz, Lt)
    static bool tile_ok(const lgt_ctx* c) {
        const Geom& g = c->g;
        return g.s_begin == 0 && g.s_end == g.V && (g.L[0] * g.L[1]) % 64 == 0 && g.L[2] % 2 == 0 && g.L[3] % 2 == 0;
    }
    // blocks (= partials) of the stencil kernels' CG modes
    static int dslash_partials(const lgt_ctx* c) {
        return (c->variant[LGT_K_DSLASH] == 3 && tile_ok(c)) ? c->g.V / 256 : site_blocks(c, 128);
    }
    // Variant 1 of LGT_K_CG_BLAS: the scalar updates of the CG loop ride in the last block of the stencil kernels
    // (cg_fused_tail) instead of two one-block launches per iteration.  Only the one-block-per-chunk kernels have the
    // tail, and the slabs of a decomposed lattice split their sums around an all-reduce.
    static unsigned* fuse_counter(const lgt_ctx* c) {
        const int dv = c->variant[LGT_K_DSLASH];
        return (c->variant[LGT_K_CG_BLAS] == 1 && !c->dd_links_valid && dv != 1 && dv != 2 && dv != 3 && dv != 9 && dv != 10 && dv != 11) ? c->counter : nullptr;
    }
    // The one-launch cooperative CG (variant 2 of LGT_K_CG_BLAS; default up to two waves of blocks): undivided lattices only
    static bool coop_wanted(const lgt_ctx* c, int nchunks) {
        if (c->dd_links_valid) return false;
        const int v = c->variant[LGT_K_CG_BLAS];
        return v == 2 || (v == 0 && c->coop_default && nchunks <= 4 * c->num_sms);
    }
    // Folded scalar updates of the even/odd CG (LGT_K_CG_BLAS variant 3): undivided lattices whose half field is at most
    // FOLD_MAX_CHUNKS blocks -- every block of the x, p update sums that many partials itself.
    static constexpr int FOLD_MAX_CHUNKS = 2048;
    static bool fold_wanted(const lgt_ctx* c, int nchunks) {
        if (c->dd_links_valid || c->g.z_hi - c->g.z_lo != c->g.L[2] || nchunks > FOLD_MAX_CHUNKS) return false;
        const int v = c->variant[LGT_K_CG_BLAS];
        return v == 3 || (v == 0 && c->fold_default);
    }
    // mode 0: out = D in / D^dag in; 1: CG "t = D p" (+ pAp, alpha); 2: CG "q = D^dag t" fused with the x, r update
    static int dslash(lgt_ctx* c, const void* U, const void* in, void* out, int dagger, int mode, void* r = nullptr,
                      const PushTo<T>* push = nullptr) {
        const int grid = site_blocks(c, 128);
        const T kappa = (T)c->kappa;
#define DSLASH_ARGS c->g, (const T2*)U, (const T2*)in, (T2*)out, kappa, c->st, c->partials, (T2*)r, PushTo<T>()
#define DSLASH_PUSH_ARGS c->g, (const T2*)U, (const T2*)in, (T2*)out, kappa, c->st, c->partials, (T2*)r, *push
        if (push && mode == 1) {  // one target, or two when push->b is set
            if (push->b) LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 2>), grid, 128, DSLASH_PUSH_ARGS);
            else LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 1>), grid, 128, DSLASH_PUSH_ARGS);
            return LGT_OK;
        }
        if (push && mode == 2) {
            if (push->b) LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 2>), grid, 128, DSLASH_PUSH_ARGS);
            else LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 1>), grid, 128, DSLASH_PUSH_ARGS);
            return LGT_OK;
        }
#undef DSLASH_PUSH_ARGS
        if (c->g.z_hi - c->g.z_lo != c->g.L[2]) {  // a rank of a (Pt, Pz) grid: the kernel that skips the ghost z planes
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 0, 1>), grid, 128, DSLASH_ARGS);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 0, 1>), grid, 128, DSLASH_ARGS);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 0, 1>), grid, 128, DSLASH_ARGS);
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 0, 1>), grid, 128, DSLASH_ARGS);
            }
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 11) {  // two chunks per block as straight-line code
            const int g2 = (grid + 1) / 2;
#define DSLASH_2ARGS c->g, (const T2*)U, (const T2*)in, (T2*)out, kappa, c->st, c->partials, (T2*)r, grid
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_two_kernel<T, 1, 0>), g2, 128, DSLASH_2ARGS);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_two_kernel<T, 0, 0>), g2, 128, DSLASH_2ARGS);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_two_kernel<T, 0, 1>), g2, 128, DSLASH_2ARGS);
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_two_kernel<T, 1, 2>), g2, 128, DSLASH_2ARGS);
            }
#undef DSLASH_2ARGS
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 10) {  // variant 1 with the chunks drawn from a counter instead of a fixed stride
            const int pgrid = grid < 2 * c->num_sms ? grid : 2 * c->num_sms;
            if (!c->coop_counter) {
                CU(cudaMalloc(&c->coop_counter, sizeof(unsigned)));
                CU(cudaMemsetAsync(c->coop_counter, 0, sizeof(unsigned), c->stream));
            }
#define DSLASH_DARGS c->g, (const T2*)U, (const T2*)in, (T2*)out, kappa, c->st, c->partials, (T2*)r, grid, c->coop_counter
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_persistent_kernel<T, 1, 0>), pgrid, 128, DSLASH_DARGS);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_persistent_kernel<T, 0, 0>), pgrid, 128, DSLASH_DARGS);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_persistent_kernel<T, 0, 1>), pgrid, 128, DSLASH_DARGS);
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_persistent_kernel<T, 1, 2>), pgrid, 128, DSLASH_DARGS);
            }
#undef DSLASH_DARGS
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 1) {  // persistent, software-pipelined: one wave of blocks loops over the chunks
            const int pgrid = grid < 2 * c->num_sms ? grid : 2 * c->num_sms;
#define DSLASH_PARGS c->g, (const T2*)U, (const T2*)in, (T2*)out, kappa, c->st, c->partials, (T2*)r, grid
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_persistent_kernel<T, 1, 0>), pgrid, 128, DSLASH_PARGS);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_persistent_kernel<T, 0, 0>), pgrid, 128, DSLASH_PARGS);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_persistent_kernel<T, 0, 1>), pgrid, 128, DSLASH_PARGS);
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_persistent_kernel<T, 1, 2>), pgrid, 128, DSLASH_PARGS);
            }
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 2) {  // persistent, forward links by bulk copy into per-warp shared-memory slots
            const int pgrid = grid < 2 * c->num_sms ? grid : 2 * c->num_sms;
            constexpr int smem = dslash_tma_smem_bytes<T>();
            if (mode == 0) {
                if (dagger)
                    LAUNCH_SMEM(c, LGT_K_DSLASH, (dslash_tma_kernel<T, 1, 0>), pgrid, 128, smem, DSLASH_PARGS);
                else
                    LAUNCH_SMEM(c, LGT_K_DSLASH, (dslash_tma_kernel<T, 0, 0>), pgrid, 128, smem, DSLASH_PARGS);
            } else if (mode == 1) {
                LAUNCH_SMEM(c, LGT_K_DSLASH, (dslash_tma_kernel<T, 0, 1>), pgrid, 128, smem, DSLASH_PARGS);
            } else {
                LAUNCH_SMEM(c, LGT_K_DSLASH_R, (dslash_tma_kernel<T, 1, 2>), pgrid, 128, smem, DSLASH_PARGS);
            }
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 9) {  // persistent, DRAM-bound operands by per-thread cp.async one chunk ahead
            const int pgrid = grid < 2 * c->num_sms ? grid : 2 * c->num_sms;
            constexpr int smem = dslash_cpasync_smem_bytes<T>();
            if (mode == 0) {
                if (dagger)
                    LAUNCH_SMEM(c, LGT_K_DSLASH, (dslash_cpasync_kernel<T, 1, 0>), pgrid, 128, smem, DSLASH_PARGS);
                else
                    LAUNCH_SMEM(c, LGT_K_DSLASH, (dslash_cpasync_kernel<T, 0, 0>), pgrid, 128, smem, DSLASH_PARGS);
            } else if (mode == 1) {
                LAUNCH_SMEM(c, LGT_K_DSLASH, (dslash_cpasync_kernel<T, 0, 1>), pgrid, 128, smem, DSLASH_PARGS);
            } else {
                LAUNCH_SMEM(c, LGT_K_DSLASH_R, (dslash_cpasync_kernel<T, 1, 2>), pgrid, 128, smem, DSLASH_PARGS);
            }
            return LGT_OK;
        }
#undef DSLASH_PARGS
        if (c->variant[LGT_K_DSLASH] == 3 && tile_ok(c)) {  // 2 x 2 x 2 tiles of 32-site layout blocks per 256-thread block
            const int tgrid = c->g.V / 256;
#define DSLASH_TARGS c->g, (const T2*)U, (const T2*)in, (T2*)out, kappa, c->st, c->partials, (T2*)r
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_tile_kernel<T, 1, 0>), tgrid, 256, DSLASH_TARGS);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_tile_kernel<T, 0, 0>), tgrid, 256, DSLASH_TARGS);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_tile_kernel<T, 0, 1>), tgrid, 256, DSLASH_TARGS);
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_tile_kernel<T, 1, 2>), tgrid, 256, DSLASH_TARGS);
            }
#undef DSLASH_TARGS
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 4) {  // variant 0 with an L2 prefetch for the block that will take this block's place
            const int pf = 2 * c->num_sms;
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 1>), grid, 128, DSLASH_ARGS, pf);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 1>), grid, 128, DSLASH_ARGS, pf);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 1>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 1>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            }
            return LGT_OK;
        }
        // Variant 8: variant 4's prefetch issued at the end of the block instead of its start.  It is also what the DEFAULT
        // (variant 0) means for the fp32 kernels on lattices of one wave of blocks up to 16384 chunks: bitwise the same
        // results, 4 - 10 % per fp32 CG iteration (16^4 ... 32^4; the inner solve of the mixed-precision solver), nothing in fp64.
        const bool late_pf = c->variant[LGT_K_DSLASH] == 8 ||
                             (c->variant[LGT_K_DSLASH] == 0 && sizeof(T) == 4 && grid > 2 * c->num_sms);
        if constexpr (sizeof(T) == 4) if (late_pf && c->variant[LGT_K_DSLASH] == 0) {  // the fp32 default: also compiled for three blocks per SM
            const int pf = 3 * c->num_sms;
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 5, 0, 1>), grid, 128, DSLASH_ARGS, pf);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 5, 0, 1>), grid, 128, DSLASH_ARGS, pf);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 5, 0, 1>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 5, 0, 1>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            }
            return LGT_OK;
        }
        if (late_pf) {
            const int pf = 2 * c->num_sms;
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 5>), grid, 128, DSLASH_ARGS, pf);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 5>), grid, 128, DSLASH_ARGS, pf);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 5>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 5>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            }
            return LGT_OK;
        }
        // Variant 12 (fp32 only; fp64 runs variant 7): 12-real links in the fp32 default's build -- three blocks per SM and the
        // end-of-block prefetch, of rows 0 and 1 only
        if constexpr (sizeof(T) == 4) if (c->variant[LGT_K_DSLASH] == 12) {
            const int pf = 3 * c->num_sms;
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 6, 0, 1>), grid, 128, DSLASH_ARGS, pf);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 6, 0, 1>), grid, 128, DSLASH_ARGS, pf);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 6, 0, 1>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 6, 0, 1>), grid, 128, DSLASH_ARGS, pf, fuse_counter(c));
            }
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 7 || c->variant[LGT_K_DSLASH] == 12) {  // 12-real links: rows 0 and 1 read, row 2 rebuilt in registers
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 4>), grid, 128, DSLASH_ARGS, 0);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 4>), grid, 128, DSLASH_ARGS, 0);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 4>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 4>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
            }
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 6) {  // variant 0 with the DRAM-bound hops (t+, z+, y+, x+) first
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 3>), grid, 128, DSLASH_ARGS, 0);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 3>), grid, 128, DSLASH_ARGS, 0);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 3>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 3>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
            }
            return LGT_OK;
        }
        if (c->variant[LGT_K_DSLASH] == 5) {  // variant 0 with the z and t neighbours loaded past L1
            if (mode == 0) {
                if (dagger)
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0, 0, 2>), grid, 128, DSLASH_ARGS, 0);
                else
                    LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0, 0, 2>), grid, 128, DSLASH_ARGS, 0);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1, 0, 2>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2, 0, 2>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
            }
            return LGT_OK;
        }
        if (mode == 0) {
            if (dagger)
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 1, 0>), grid, 128, DSLASH_ARGS);
            else
                LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 0>), grid, 128, DSLASH_ARGS);
        } else if (mode == 1) {
            LAUNCH(c, LGT_K_DSLASH, (dslash_kernel<T, 0, 1>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
        } else {
            LAUNCH(c, LGT_K_DSLASH_R, (dslash_kernel<T, 1, 2>), grid, 128, DSLASH_ARGS, 0, fuse_counter(c));
        }
#undef DSLASH_ARGS
        return LGT_OK;
    }

    // CG on D^dag D (reading A-10): b, x native; y (optional) receives D x.
    // Per iteration: t = D p (+ |t|^2) | alpha | q = D^dag t fused with r -= alpha q (+ |r|^2) | beta, stop test |
    // x += alpha p, p = r + beta p.
    // U: native links of precision T; wr, wp, wt: three native spinor workspaces of precision T.
    static int cg(lgt_ctx* c, const void* U, void* wr, void* wp, void* wt, const void* b, void* x, void* y, double tol,
                  int max_iter, int* iters, double* rel, double pcoef = 0.0) {
        T2 *r = (T2*)wr, *p = (T2*)wp, *t = (T2*)wt;
        const size_t n = (size_t)12 * c->g.Vs;
        const int nb = stream_blocks(c, n);
        const int ngrid = dslash_partials(c);  // blocks (= partials) of the stencil kernels
        const bool fused = fuse_counter(c) != nullptr;
        LAUNCH(c, LGT_K_CG_BLAS, (cg_init_kernel<T>), nb, 256, n, (const T2*)b, (T2*)x, r, p, c->st, tol * tol, max_iter, c->partials, c->counter, ZMask(), (T)pcoef);
        int rc;
        int launched = 0;
        for (;;) {
            CU(cudaMemcpyAsync(c->h_st, c->st, sizeof(CgState), cudaMemcpyDeviceToHost, c->stream));
            CU(cudaStreamSynchronize(c->stream));
            if (c->h_st->done) break;
            // iterations are enqueued in chunks; kernels past convergence return at once
            int chunk = max_iter - launched;
            if (chunk > 8) chunk = 8;
            if (chunk <= 0) chunk = 1;
            auto body = [&]() -> int {
                int r2;
                for (int i = 0; i < chunk; i++) {
                    if ((r2 = dslash(c, U, p, t, 0, 1)) != LGT_OK) return r2;
                    if (!fused) LAUNCH(c, LGT_K_CG_BLAS, (cg_scalars_kernel<1>), 1, 1024, ngrid, c->partials, c->st);
                    if ((r2 = dslash(c, U, t, nullptr, 1, 2, r)) != LGT_OK) return r2;
                    if (!fused) LAUNCH(c, LGT_K_CG_BLAS, (cg_scalars_kernel<2>), 1, 1024, ngrid, c->partials, c->st);
                    LAUNCH(c, LGT_K_CG_UPDATE, (cg_update_xp_kernel<T>), nb, 256, n, (T2*)x, p, (const T2*)r, c->st);
                }
                return LGT_OK;
            };
            const void* const key[7] = {U, x, r, p, t, (const void*)(size_t)fused, (const void*)sizeof(T)};
            if ((rc = (chunk == 8 ? chunk_graph(c, 0, key, body) : body())) != LGT_OK) return rc;
            launched += chunk;
        }
        const CgState& h = *c->h_st;
        if (iters) *iters = h.iter;
        if (rel) *rel = (h.bb > 0.0) ? sqrt(h.rr / h.bb) : 0.0;
        if (y && (rc = dslash(c, U, x, y, 0, 0)) != LGT_OK) return rc;
        if (h.rr > h.tol2 * h.bb) return fail(c, LGT_ENOCONV, "CG did not reach the tolerance within max_iter");
        return LGT_OK;
    }

    // ---- stout smearing: the Dirac operator sees c->Uf
    // Brings c->Uf up to date: the thin links, or level nsmear of U^(k+1) = exp(A^(k+1)) U^(k), A = -rho P_su(3)[U V].
    static int smear_alloc(lgt_ctx* c) {
        for (int k = 0; k < c->nsmear; k++) {
            if (!c->Usm[k]) CU(cudaMalloc(&c->Usm[k], links_bytes(c)));
            if (!c->Asm[k]) {
                CU(cudaMalloc(&c->Asm[k], mom_bytes(c)));
                CU(cudaMemsetAsync(c->Asm[k], 0, mom_bytes(c), c->stream));
            }
        }
        return LGT_OK;
    }
    // level k + 1 from level k (the owned sites; on a slab the caller exchanges the ghost slices of the result)
    static int smear_level(lgt_ctx* c, int k) {
        const int grid = site_blocks(c, 32);
        const T2* Uin = (const T2*)(k == 0 ? c->U : c->Usm[k - 1]);
        if (c->g.Vs != c->g.V) CU(cudaMemsetAsync(c->Usm[k], 0, links_bytes(c), c->stream));  // padding lanes
        LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_kernel<T, 0>), grid, 128, c->g, Uin, (T2*)c->Asm[k], (T)(-c->rho), (T)0);
        LAUNCH(c, LGT_K_LINK_UPDATE, (link_update_kernel<T>), grid, 128, c->g, Uin, (T2*)c->Usm[k], (const T2*)c->Asm[k], (T)1);
        return LGT_OK;
    }
    static int ensure_fermion_links(lgt_ctx* c) {
        if (c->nsmear == 0) {
            c->Uf = c->U;
            return LGT_OK;
        }
        int rc;
        if ((rc = smear_alloc(c)) != LGT_OK) return rc;
        if (!c->usm_valid && !c->dd_links_valid) {  // on a slab the group driver interleaves the levels with halo exchanges
            for (int k = 0; k < c->nsmear; k++)
                if ((rc = smear_level(c, k)) != LGT_OK) return rc;
            c->usm_valid = true;
        }
        c->Uf = c->Usm[c->nsmear - 1];
        return LGT_OK;
    }

    // F^f from X, Y: Pi -= eps F (acc) or F written to P (compact).  With smearing, the force with respect to the
    // smeared links is pulled back level by level (stout_local_kernel, stout_chain_kernel) to the thin links.
    static int fermion_force(lgt_ctx* c, const void* X, const void* Y, void* P, int acc, double eps) {
        int rc;
        if ((rc = ensure_fermion_links(c)) != LGT_OK) return rc;
        const int grid = site_blocks(c, 128);
        if (c->nsmear == 0) {
            if (acc)
                LAUNCH(c, LGT_K_FERMION_FORCE, (fermion_force_kernel<T, 1>), grid, 128, c->g, (const T2*)c->Uf, (const T2*)X, (const T2*)Y, (T2*)P, (T)c->kappa, (T)eps);
            else
                LAUNCH(c, LGT_K_FERMION_FORCE, (fermion_force_kernel<T, 0>), grid, 128, c->g, (const T2*)c->Uf, (const T2*)X, (const T2*)Y, (T2*)P, (T)c->kappa, (T)eps);
            return LGT_OK;
        }
        if (!c->F2) {
            CU(cudaMalloc(&c->F2, mom_bytes(c)));
            CU(cudaMalloc(&c->F3, mom_bytes(c)));
            CU(cudaMalloc(&c->F4, mom_bytes(c)));
            CU(cudaMemsetAsync(c->F2, 0, mom_bytes(c), c->stream));
            CU(cudaMemsetAsync(c->F3, 0, mom_bytes(c), c->stream));
            CU(cudaMemsetAsync(c->F4, 0, mom_bytes(c), c->stream));
        }
        const int lgrid = site_blocks(c, 32);
        T2 *Fa = (T2*)c->F3, *Fb = (T2*)c->F4, *G = (T2*)c->F2;  // P is never one of these
        LAUNCH(c, LGT_K_FERMION_FORCE, (fermion_force_kernel<T, 0>), grid, 128, c->g, (const T2*)c->Uf, (const T2*)X, (const T2*)Y, Fa, (T)c->kappa, (T)0);
        for (int k = c->nsmear - 1; k >= 0; k--) {
            const T2* Uk = (const T2*)(k == 0 ? c->U : c->Usm[k - 1]);
            LAUNCH(c, LGT_K_FERMION_FORCE, (stout_local_kernel<T>), lgrid, 128, c->g, (const T2*)c->Asm[k], Fa, G);
            if (k == 0 && acc)
                LAUNCH(c, LGT_K_FERMION_FORCE, (stout_chain_kernel<T, 1>), lgrid, 128, c->g, Uk, (const T2*)G, (const T2*)Fa, (T2*)P, (T)c->rho, (T)eps);
            else
                LAUNCH(c, LGT_K_FERMION_FORCE, (stout_chain_kernel<T, 0>), lgrid, 128, c->g, Uk, (const T2*)G, (const T2*)Fa, (k == 0 ? (T2*)P : Fb), (T)c->rho, (T)0);
            T2* t = Fa;
            Fa = Fb;
            Fb = t;
        }
        return LGT_OK;
    }
    static int gauge_force(lgt_ctx* c, void* P, int acc, double eps) {
        const int grid = site_blocks(c, 32);
        const int v = c->variant[LGT_K_GAUGE_FORCE];
        if (v == 3) {  // one thread per site, up staples plaquette by plaquette
            const int g1 = site_blocks(c, 128);
            if (acc) LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_site_kernel<T, 1>), g1, 128, c->g, (const T2*)c->U, (T2*)P, (T)(c->beta / 6.0), (T)eps);
            else LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_site_kernel<T, 0>), g1, 128, c->g, (const T2*)c->U, (T2*)P, (T)(c->beta / 6.0), (T)eps);
            return LGT_OK;
        }
        if (v == 1 || v == 2) {  // 2 / 4 layout blocks per thread block
            const int rows = 2 * v, g4 = site_blocks(c, 128) * (4 / rows);
#define GF_ARGS c->g, (const T2*)c->U, (T2*)P, (T)(c->beta / 6.0), (T)eps
            if (v == 1) {
                if (acc) LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_kernel<T, 1, 2>), g4, 256, GF_ARGS);
                else LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_kernel<T, 0, 2>), g4, 256, GF_ARGS);
            } else {
                if (acc) LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_kernel<T, 1, 4>), g4, 512, GF_ARGS);
                else LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_kernel<T, 0, 4>), g4, 512, GF_ARGS);
            }
#undef GF_ARGS
            return LGT_OK;
        }
        if (acc)
            LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_kernel<T, 1>), grid, 128, c->g, (const T2*)c->U, (T2*)P, (T)(c->beta / 6.0), (T)eps);
        else
            LAUNCH(c, LGT_K_GAUGE_FORCE, (gauge_force_kernel<T, 0>), grid, 128, c->g, (const T2*)c->U, (T2*)P, (T)(c->beta / 6.0), (T)eps);
        return LGT_OK;
    }
    static int link_update(lgt_ctx* c, double eps) {
        const int grid = site_blocks(c, 32);
        c->u32_valid = false;
    c->usm_valid = false;
    if (c->dd_links_valid) *c->dd_links_valid = false;
        c->ucb_valid = false;
    c->ucb32_valid = false;
    c->inner_exact = false;
        p_ready(c);
        LAUNCH(c, LGT_K_LINK_UPDATE, (link_update_kernel<T>), grid, 128, c->g, (const T2*)c->U, (T2*)c->U, (const T2*)c->P, (T)eps);
        return LGT_OK;
    }
    static int plaquette_sum(lgt_ctx* c, double* dev_result) {
        LAUNCH(c, LGT_K_OTHER, (plaquette_kernel<T>), site_blocks(c, 128), 128, c->g, (const T2*)c->U, dev_result, c->partials, c->counter);
        return LGT_OK;
    }
    static int kinetic(lgt_ctx* c, double* dev_result) {
        p_ready(c);
        LAUNCH(c, LGT_K_OTHER, (kinetic_kernel<T>), stream_blocks(c, (size_t)4 * c->g.Vs), 256, c->g, (const T2*)c->P, dev_result, c->partials, c->counter);
        return LGT_OK;
    }
    static int redot(lgt_ctx* c, const void* a, const void* b, double* dev_result, size_t n = 0) {
        if (n == 0) n = (size_t)12 * c->g.Vs;
        LAUNCH(c, LGT_K_OTHER, (redot_kernel<T>), stream_blocks(c, n), 256, n, (const T2*)a, (const T2*)b, dev_result, c->partials, c->counter);
        return LGT_OK;
    }

    static int momentum_heatbath(lgt_ctx* c, unsigned long long seed, unsigned traj) {
        p_ready(c);
        LAUNCH(c, LGT_K_OTHER, (momentum_heatbath_kernel<T>), stream_blocks(c, (size_t)4 * c->g.Vs), 256, c->g, (T2*)c->P, seed, traj);
        return LGT_OK;
    }
    // eta ~ exp(-eta^dag eta) into ws[4]; phi = D^dag eta (full action) or phi_e = M^dag eta_e (even/odd action);
    // S_F at the start of the trajectory, |eta|^2 resp. |eta_e|^2, to dev_SF0.
    static int pseudofermion_heatbath(lgt_ctx* c, unsigned long long seed, unsigned traj, double* dev_SF0) {
        int rc;
        if ((rc = ensure_fermion_links(c)) != LGT_OK) return rc;
        T2* eta = (T2*)c->ws[4];
        LAUNCH(c, LGT_K_OTHER, (spinor_heatbath_kernel<T>), stream_blocks(c, (size_t)12 * c->g.Vs), 256, c->g, eta, seed, traj);
        if (c->action == LGT_ACTION_EO) {
            if ((rc = eo_ensure(c)) != LGT_OK) return rc;
            if ((rc = eo_split(c, eta, eo_field(c, 4))) != LGT_OK) return rc;  // fields 4, 5 = (eta_e, eta_o)
            if ((rc = eo_mhat(c, eo_field(c, 4), eo_field(c, 2), eo_field(c, 7), 1)) != LGT_OK) return rc;
            CU(cudaMemsetAsync(eo_field(c, 3), 0, (size_t)12 * c->g.Vhs * sizeof(T2), c->stream));
            if ((rc = eo_merge(c, eo_field(c, 2), c->phi)) != LGT_OK) return rc;
            if (dev_SF0 && (rc = redot(c, eo_field(c, 4), eo_field(c, 4), dev_SF0, (size_t)12 * c->g.Vhs)) != LGT_OK) return rc;
        } else {
            if ((rc = dslash(c, c->Uf, eta, c->phi, 1, 0)) != LGT_OK) return rc;
            if (dev_SF0 && (rc = redot(c, eta, eta, dev_SF0, 0)) != LGT_OK) return rc;
        }
        c->has_phi = true;
        return LGT_OK;
    }

    // ---- even/odd preconditioning
    // Ops<float> on an LGT_F64 handle (the fp32 inner solve of the mixed-precision solver) works on the fp32 copies
    static bool fp32_on_f64(const lgt_ctx* c) { return sizeof(T) == 4 && c->prec == LGT_F64; }
    static T2* eo_field(lgt_ctx* c, int i) { return (T2*)(fp32_on_f64(c) ? c->eo32 : c->eo) + (size_t)i * 12 * c->g.Vhs; }
    static const T2* links_cb(lgt_ctx* c, int p) { return (const T2*)(fp32_on_f64(c) ? c->Ucb32 : c->Ucb) + (size_t)p * 36 * c->g.Vhs; }
    static int eo_ensure(lgt_ctx* c) {
        int rcf = ensure_fermion_links(c);
        if (rcf != LGT_OK) return rcf;
        if (!c->Ucb) {
            CU(cudaMalloc(&c->Ucb, (size_t)2 * 36 * c->g.Vhs * sizeof(T2)));
            c->ucb_valid = false;
    c->ucb32_valid = false;
    c->inner_exact = false;
        }
        if (!c->eo) {
            CU(cudaMalloc(&c->eo, (size_t)8 * 12 * c->g.Vhs * sizeof(T2)));
            CU(cudaMemsetAsync(c->eo, 0, (size_t)8 * 12 * c->g.Vhs * sizeof(T2), c->stream));
        }
        if (!c->ucb_valid) {
            const size_t n = (size_t)2 * 36 * c->g.Vhs;
            LAUNCH(c, LGT_K_OTHER, (eo_reorder_kernel<T, 0, 36>), stream_blocks(c, n), 256, c->g, (T2*)c->Uf, (T2*)c->Ucb);
            c->ucb_valid = true;
        }
        return LGT_OK;
    }
    // full native spinor -> (even, odd) halves at eo fields (ie, ie + 1), or back
    static int eo_split(lgt_ctx* c, const void* full, T2* halves) {
        const size_t n = (size_t)2 * 12 * c->g.Vhs;
        LAUNCH(c, LGT_K_OTHER, (eo_reorder_kernel<T, 0, 12>), stream_blocks(c, n), 256, c->g, (T2*)full, halves);
        return LGT_OK;
    }
    static int eo_merge(lgt_ctx* c, T2* halves, void* full) {
        const size_t n = (size_t)2 * 12 * c->g.Vhs;
        LAUNCH(c, LGT_K_OTHER, (eo_reorder_kernel<T, 1, 12>), stream_blocks(c, n), 256, c->g, (T2*)full, halves);
        return LGT_OK;
    }
    // out (parity p) = self - kap * H in (in of parity 1 - p); mode as in hop_cb_kernel
    static int hop(lgt_ctx* c, int p, const T2* in, const T2* self, T2* out, int dagger, int mode, double kap, T2* r = nullptr,
                   const PushTo<T>* push = nullptr) {
        const int grid = (own_half_sites(c) + 127) / 128;
#define HOP_PUSH_ARGS c->g, p, links_cb(c, p), links_cb(c, 1 - p), in, self, out, (T)kap, c->st, c->partials, r, *push
        if (push && mode == 1) {
            if (push->b) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 1, 2>), grid, 128, HOP_PUSH_ARGS);
            else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 1, 1>), grid, 128, HOP_PUSH_ARGS);
            return LGT_OK;
        }
        if (push && mode == 2) {
            if (push->b) LAUNCH(c, LGT_K_DSLASH_R, (hop_cb_kernel<T, 1, 2, 2>), grid, 128, HOP_PUSH_ARGS);
            else LAUNCH(c, LGT_K_DSLASH_R, (hop_cb_kernel<T, 1, 2, 1>), grid, 128, HOP_PUSH_ARGS);
            return LGT_OK;
        }
#undef HOP_PUSH_ARGS
#define HOP_ARGS c->g, p, links_cb(c, p), links_cb(c, 1 - p), in, self, out, (T)kap, c->st, c->partials, r, PushTo<T>()
        if (c->g.z_hi - c->g.z_lo != c->g.L[2]) {  // a rank of a (Pt, Pz) grid: the kernels that skip the ghost z planes
            if (mode == 0) {
                if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 0, 0, 1>), grid, 128, HOP_ARGS);
                else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 0, 0, 1>), grid, 128, HOP_ARGS);
            } else if (mode == 3) {
                if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 3, 0, 1>), grid, 128, HOP_ARGS);
                else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 3, 0, 1>), grid, 128, HOP_ARGS);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 1, 0, 1>), grid, 128, HOP_ARGS);
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (hop_cb_kernel<T, 1, 2, 0, 1>), grid, 128, HOP_ARGS);
            }
            return LGT_OK;
        }
        // (time slabs of a decomposed lattice take it too: the prefetch never leaves [h_begin, h_end), the folded sign knows the slab's offset)
        if (sizeof(T) == 4 && (c->variant[LGT_K_DSLASH] == 0 || c->variant[LGT_K_DSLASH] == 12) && grid > 2 * c->num_sms) {
            // the fp32 hops with the end-of-block L2 prefetch for the block that takes this block's place (as the fp32 Dslash default);
            // PFL 2: the same build with 12-real links -- rows 0 and 1 of every link read, row 2 rebuilt in registers.  These
            // kernels ARE bound by bytes (0.95 of the copy bandwidth), so the 192 B per site less pay: 32^4 hop 67 -> 59 us, the
            // even/odd mixed-precision MD step 27.9 -> 25.4 ms at the same iteration count.  It is the default where it cannot
            // change an answer: in the fp32 INNER solve of the mixed-precision solver, whose result the fp64 defect correction
            // checks against the exact operator (links that are not special unitary would cost iterations, not accuracy).  A
            // plain fp32 handle keeps the exact 9-entry links unless variant 12 of LGT_K_DSLASH is selected.
            const bool twelve = c->variant[LGT_K_DSLASH] == 12 || (fp32_on_f64(c) && !c->inner_exact);
            const int pf = 2 * c->num_sms;
            auto launch_pfl = [&](auto tag) -> int {
                constexpr int PF = decltype(tag)::value;
                if (mode == 0) {
                    if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 0, 0, 0, PF>), grid, 128, HOP_ARGS, nullptr, pf);
                    else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 0, 0, 0, PF>), grid, 128, HOP_ARGS, nullptr, pf);
                } else if (mode == 3) {
                    if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 3, 0, 0, PF>), grid, 128, HOP_ARGS, nullptr, pf);
                    else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 3, 0, 0, PF>), grid, 128, HOP_ARGS, nullptr, pf);
                } else if (mode == 4) {  // mode 3 + the alpha duty of the folded scalar updates (D^dag half only)
                    LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 4, 0, 0, PF>), grid, 128, HOP_ARGS, nullptr, pf, grid);
                } else if (mode == 1) {
                    LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 1, 0, 0, PF>), grid, 128, HOP_ARGS, fuse_counter(c), pf);
                } else {
                    LAUNCH(c, LGT_K_DSLASH_R, (hop_cb_kernel<T, 1, 2, 0, 0, PF>), grid, 128, HOP_ARGS, fuse_counter(c), pf);
                }
                return LGT_OK;
            };
            if constexpr (sizeof(T) == 4) {
                return twelve ? launch_pfl(std::integral_constant<int, 2>()) : launch_pfl(std::integral_constant<int, 1>());
            }
        }
        if constexpr (sizeof(T) == 8) if (c->variant[LGT_K_DSLASH] == 12) {  // fp64 hops on 12-real links (opt-in: exact for special unitary links only)
            if (mode == 0) {
                if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 0, 0, 0, 4>), grid, 128, HOP_ARGS);
                else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 0, 0, 0, 4>), grid, 128, HOP_ARGS);
            } else if (mode == 3) {
                if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 3, 0, 0, 4>), grid, 128, HOP_ARGS);
                else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 3, 0, 0, 4>), grid, 128, HOP_ARGS);
            } else if (mode == 4) {
                LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 4, 0, 0, 4>), grid, 128, HOP_ARGS, nullptr, 0, grid);
            } else if (mode == 1) {
                LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 1, 0, 0, 4>), grid, 128, HOP_ARGS, fuse_counter(c));
            } else {
                LAUNCH(c, LGT_K_DSLASH_R, (hop_cb_kernel<T, 1, 2, 0, 0, 4>), grid, 128, HOP_ARGS, fuse_counter(c));
            }
            return LGT_OK;
        }
        if (mode == 0) {
            if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 0>), grid, 128, HOP_ARGS);
            else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 0>), grid, 128, HOP_ARGS);
        } else if (mode == 3) {
            if (dagger) LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 3>), grid, 128, HOP_ARGS);
            else LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 3>), grid, 128, HOP_ARGS);
        } else if (mode == 4) {
            LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 1, 4>), grid, 128, HOP_ARGS, nullptr, 0, grid);
        } else if (mode == 1) {
            LAUNCH(c, LGT_K_DSLASH, (hop_cb_kernel<T, 0, 1>), grid, 128, HOP_ARGS, fuse_counter(c));
        } else {
            LAUNCH(c, LGT_K_DSLASH_R, (hop_cb_kernel<T, 1, 2>), grid, 128, HOP_ARGS, fuse_counter(c));
        }
#undef HOP_ARGS
        return LGT_OK;
    }
    // out_e = M in_e (dagger: M^dag in_e), M = 1 - kappa^2 H_eo H_oe; scratch_o receives kappa H_oe in_e
    static int eo_mhat(lgt_ctx* c, const T2* in_e, T2* out_e, T2* scratch_o, int dagger) {
        int rc;
        if ((rc = hop(c, 1, in_e, nullptr, scratch_o, dagger, 0, -c->kappa)) != LGT_OK) return rc;
        return hop(c, 0, scratch_o, in_e, out_e, dagger, 0, c->kappa);
    }
    // CG on M^dag M x_e = b_e, x0 = 0, same recurrence and stop rule as cg(); u_e, t_o are scratch half fields.
    // pcoef != 0: p = b + pcoef p instead of p = b at the start (the previous solve's search direction is kept; eo_cg_mixed)
    static int eo_cg(lgt_ctx* c, const T2* b, T2* x, T2* r, T2* p, T2* u, T2* t, double tol, int max_iter, int* iters, double* rel,
                     double pcoef = 0.0) {
        const size_t n = (size_t)12 * c->g.Vhs;
        const int nb = stream_blocks(c, n);
        const int ngrid = (own_half_sites(c) + 127) / 128;
        const bool fused = fuse_counter(c) != nullptr;
        LAUNCH(c, LGT_K_CG_BLAS, (cg_init_kernel<T>), nb, 256, n, b, x, r, p, c->st, tol * tol, max_iter, c->partials, c->counter, ZMask(), (T)pcoef);
        int rc, launched = 0;
        // Small lattices: the whole solve in one cooperative launch (eo_cg_coop_kernel; LGT_K_CG_BLAS variant 2, and the
        // default while the half field is at most two waves of blocks).  Bitwise the iterates of the loop below.
        if (coop_wanted(c, ngrid)) {
            int per_sm = 0;
            CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, eo_cg_coop_kernel<T>, 128, 0));
            int cgrid = per_sm * c->num_sms;
            if (cgrid > ngrid) cgrid = ngrid;
            if (cgrid >= 1) {
                if (!c->coop_counter) {
                    CU(cudaMalloc(&c->coop_counter, sizeof(unsigned)));
                    CU(cudaMemsetAsync(c->coop_counter, 0, sizeof(unsigned), c->stream));
                }
                Geom g = c->g;
                const T2 *U0 = links_cb(c, 0), *U1 = links_cb(c, 1);
                T kap = (T)c->kappa;
                int nch = ngrid;
                void* args[] = {&g, &U0, &U1, &x, &r, &p, &u, &t, &kap, &c->st, &c->partials, &c->coop_counter, &nch};
                cudaEvent_t e0 = nullptr, e1 = nullptr;
                if (c->timing && (e0 = timing_event(c)) && (e1 = timing_event(c))) {
                    c->ev_class.push_back(LGT_K_DSLASH);
                    cudaEventRecord(e0, c->stream);
                }
                CU(cudaLaunchCooperativeKernel((const void*)eo_cg_coop_kernel<T>, dim3(cgrid), dim3(128), args, 0, c->stream));
                if (e0 && e1) cudaEventRecord(e1, c->stream);
                c->launches++;
                CU(cudaMemcpyAsync(c->h_st, c->st, sizeof(CgState), cudaMemcpyDeviceToHost, c->stream));
                CU(cudaStreamSynchronize(c->stream));
                const CgState& hc = *c->h_st;
                if (iters) *iters = hc.iter;
                if (rel) *rel = (hc.bb > 0.0) ? sqrt(hc.rr / hc.bb) : 0.0;
                if (hc.rr > hc.tol2 * hc.bb) return fail(c, LGT_ENOCONV, "even/odd CG did not reach the tolerance within max_iter");
                return LGT_OK;
            }
        }
        // Small lattices, the scalar updates FOLDED into the kernels that follow them (LGT_K_CG_BLAS variant 3): five launches
        // per iteration instead of seven, no fence or ticket.  pAp and alpha: block 0 of the third hop (hop mode 4); |r|^2,
        // beta, count and stop test: every block of the x, p update, from the same partials in the same fixed order, block 0
        // writing the next iteration's state into the other of two CgState (cg_update_xp_fold_kernel).  Bitwise the iterates
        // of the loop below.
        if (fold_wanted(c, ngrid)) {
            CgState* const S[2] = {c->st, c->st2};
            int par = 0;
            for (;;) {
                CU(cudaMemcpyAsync(c->h_st, S[par], sizeof(CgState), cudaMemcpyDeviceToHost, c->stream));
                CU(cudaStreamSynchronize(c->stream));
                if (c->h_st->done) break;
                int chunk = max_iter - launched;
                if (chunk > 8) chunk = 8;
                if (chunk <= 0) chunk = 1;
                const int par0 = par;
                auto body = [&]() -> int {
                    int r2 = LGT_OK, q = par0;
                    for (int i = 0; i < chunk && r2 == LGT_OK; i++, q ^= 1) {
                        c->st = S[q];
                        if ((r2 = hop(c, 1, p, nullptr, t, 0, 3, -c->kappa)) != LGT_OK) break;   // t_o = kappa H_oe p
                        if ((r2 = hop(c, 0, t, p, u, 0, 1, c->kappa)) != LGT_OK) break;          // u = M p, partials of |u|^2
                        if ((r2 = hop(c, 1, u, nullptr, t, 1, 4, -c->kappa)) != LGT_OK) break;   // t_o = kappa H^dag_oe u; pAp, alpha
                        if ((r2 = hop(c, 0, t, u, nullptr, 1, 2, c->kappa, r)) != LGT_OK) break; // r -= alpha M^dag u, partials of |r|^2
                        r2 = [&]() -> int {
                            LAUNCH(c, LGT_K_CG_UPDATE, (cg_update_xp_fold_kernel<T>), nb, 256, n, x, p, (const T2*)r, (const CgState*)S[q], S[q ^ 1],
                                   (const double*)c->partials, ngrid);
                            return LGT_OK;
                        }();
                    }
                    c->st = S[0];
                    return r2;
                };
                const void* const key[7] = {links_cb(c, 0), x, r, p, u, t, (const void*)(sizeof(T) + 128)};
                if ((rc = (chunk == 8 && par == 0 ? chunk_graph(c, 1, key, body) : body())) != LGT_OK) return rc;
                launched += chunk;
                par ^= (chunk & 1);
            }
            if (par) CU(cudaMemcpyAsync(S[0], S[1], sizeof(CgState), cudaMemcpyDeviceToDevice, c->stream));
            const CgState& h = *c->h_st;
            if (iters) *iters = h.iter;
            if (rel) *rel = (h.bb > 0.0) ? sqrt(h.rr / h.bb) : 0.0;
            if (h.rr > h.tol2 * h.bb) return fail(c, LGT_ENOCONV, "even/odd CG did not reach the tolerance within max_iter");
            return LGT_OK;
        }
        for (;;) {
            CU(cudaMemcpyAsync(c->h_st, c->st, sizeof(CgState), cudaMemcpyDeviceToHost, c->stream));
            CU(cudaStreamSynchronize(c->stream));
            if (c->h_st->done) break;
            int chunk = max_iter - launched;
            if (chunk > 8) chunk = 8;
            if (chunk <= 0) chunk = 1;
            auto body = [&]() -> int {
                int r2;
                for (int i = 0; i < chunk; i++) {
                    if ((r2 = hop(c, 1, p, nullptr, t, 0, 3, -c->kappa)) != LGT_OK) return r2;   // t_o = kappa H_oe p
                    if ((r2 = hop(c, 0, t, p, u, 0, 1, c->kappa)) != LGT_OK) return r2;          // u = M p, |u|^2
                    if (!fused) LAUNCH(c, LGT_K_CG_BLAS, (cg_scalars_kernel<1>), 1, 1024, ngrid, c->partials, c->st);
                    if ((r2 = hop(c, 1, u, nullptr, t, 1, 3, -c->kappa)) != LGT_OK) return r2;   // t_o = kappa H^dag_oe u
                    if ((r2 = hop(c, 0, t, u, nullptr, 1, 2, c->kappa, r)) != LGT_OK) return r2; // r -= alpha M^dag u
                    if (!fused) LAUNCH(c, LGT_K_CG_BLAS, (cg_scalars_kernel<2>), 1, 1024, ngrid, c->partials, c->st);
                    LAUNCH(c, LGT_K_CG_UPDATE, (cg_update_xp_kernel<T>), nb, 256, n, x, p, (const T2*)r, c->st);
                }
                return LGT_OK;
            };
            const void* const key[7] = {links_cb(c, 0), x, r, p, u, t, (const void*)(sizeof(T) + 64 * (size_t)fused)};
            if ((rc = (chunk == 8 ? chunk_graph(c, 1, key, body) : body())) != LGT_OK) return rc;
            launched += chunk;
        }
        const CgState& h = *c->h_st;
        if (iters) *iters = h.iter;
        if (rel) *rel = (h.bb > 0.0) ? sqrt(h.rr / h.bb) : 0.0;
        if (h.rr > h.tol2 * h.bb) return fail(c, LGT_ENOCONV, "even/odd CG did not reach the tolerance within max_iter");
        return LGT_OK;
    }
    // Even/odd action: X_e = (M^dag M)^-1 phi_e, Y_e = M X_e, X_o = kappa H_oe X_e, Y_o = kappa H^dag_oe Y_e, merged into
    // the full fields X, Y (native) that the fused force kernel takes; Re <phi_e, X_e> to dev_SF if not null.
    static int eo_solve_xy(lgt_ctx* c, void* X, void* Y, double tol, int max_iter, int* iters, double* dev_SF) {
        int rc, conv;
        if ((rc = eo_ensure(c)) != LGT_OK) return rc;
        T2 *Xe = eo_field(c, 0), *Xo = eo_field(c, 1), *Ye = eo_field(c, 2), *Yo = eo_field(c, 3);
        T2 *be = eo_field(c, 4), *re = eo_field(c, 5), *pe = eo_field(c, 6), *to = eo_field(c, 7);
        if ((rc = eo_split(c, c->phi, be)) != LGT_OK) return rc;  // (be, re) receive (phi_e, phi_o); re is overwritten next
        // The mixed-precision solver's last true residual r = b - M^dag (M x) leaves u = M x = Y_e behind and, in the odd scratch
        // field of the M^dag application, kappa H^dag_oe u = Y_o: with Y_o as that scratch field only X_o is left to compute
        // (one fp64 hop instead of three; the same kernels on the same input, so bitwise the fields of the general path).
        bool have_y = false;
        if (c->solver == LGT_SOLVER_MIXED_CG && c->prec == LGT_F64 && sizeof(T) == 8) {
            c->last_outer = 0;
            conv = eo_cg_mixed(c, be, Xe, re, pe, Ye, Yo, tol, max_iter, iters);
            have_y = c->last_outer > 0;
        } else
            conv = eo_cg(c, be, Xe, re, pe, Ye, to, tol, max_iter, iters, nullptr);
        if (conv != LGT_OK && conv != LGT_ENOCONV) return conv;
        if (dev_SF && (rc = redot(c, be, Xe, dev_SF, (size_t)12 * c->g.Vhs)) != LGT_OK) return rc;
        if (X && Y && have_y) {
            if ((rc = hop(c, 1, Xe, nullptr, Xo, 0, 0, -c->kappa)) != LGT_OK) return rc;  // X_o = kappa H_oe X_e
            if ((rc = eo_merge(c, Xe, X)) != LGT_OK) return rc;
            if ((rc = eo_merge(c, Ye, Y)) != LGT_OK) return rc;
        } else if (X && Y) {
            if ((rc = eo_mhat(c, Xe, Ye, Xo, 0)) != LGT_OK) return rc;                  // Y_e = M X_e, X_o = kappa H_oe X_e
            if ((rc = hop(c, 1, Ye, nullptr, Yo, 1, 0, -c->kappa)) != LGT_OK) return rc;  // Y_o = kappa H^dag_oe Y_e
            if ((rc = eo_merge(c, Xe, X)) != LGT_OK) return rc;
            if ((rc = eo_merge(c, Ye, Y)) != LGT_OK) return rc;
        }
        return conv;
    }
};

#define DISPATCH(c, fn, ...) ((c)->prec == LGT_F64 ? Ops<double>::fn(__VA_ARGS__) : Ops<float>::fn(__VA_ARGS__))

int read_scalars(lgt_ctx* c, int n) {
    CU(cudaMemcpyAsync(c->h_scal, c->scal, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return LGT_OK;
}

// Mixed-precision solve of (M^dag M) x_e = b_e on an fp64 handle: the defect correction of cg_mixed() with the even/odd
// operator -- fp32 CG on the Schur complement (fp32 checkerboard links and half fields) inside, true fp64 residual
// r = b - M^dag M x outside, stop on |r| <= tol |b|.  b, x, r, q, u: fp64 even half fields; t_o: an odd scratch field.
//
// Safety net of the 12-real inner hops (hop(): PFL 2): a correction cycle that was asked for a reduction of the residual by
// eps and delivered less than a factor 100 -- and less than a tenth of what was asked -- means that the inner operator is not
// the outer one to fp32 accuracy, i.e. the links are not special unitary.  The inner hops then read the exact 9-entry links
// from here on (the flag holds until the links change; captured CG chunks are dropped, they hold the 12-real kernels).
// rr_old, rr_new: |r|^2 before and after the cycle.  Returns true if it switched.
bool mixed_inner_fallback(lgt_ctx* c, double rr_old, double rr_new, double eps) {
    if (c->inner_exact || !(rr_new > 1e-4 * rr_old && rr_new > 100.0 * eps * eps * rr_old)) return false;
    c->inner_exact = true;
    for (lgt_ctx::ChunkGraph& g : c->graphs) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
    return true;
}
int eo_cg_mixed(lgt_ctx* c, void* b, void* x, void* r, void* q, void* u, void* t_o, double tol, int max_iter, int* iters) {
    typedef Ops<double> O64;
    typedef Ops<float> O32;
    const size_t n = (size_t)12 * c->g.Vhs;
    if (!c->Ucb32) {
        CU(cudaMalloc(&c->Ucb32, (size_t)2 * 36 * c->g.Vhs * sizeof(float2)));
        CU(cudaMalloc(&c->eo32, (size_t)6 * n * sizeof(float2)));
        CU(cudaMemsetAsync(c->eo32, 0, (size_t)6 * n * sizeof(float2), c->stream));
        c->ucb32_valid = false;
        c->inner_exact = false;
    }
    const int nb = stream_blocks(c, n);
    if (!c->ucb32_valid) {
        const size_t nu = (size_t)2 * 36 * c->g.Vhs;
        LAUNCH(c, LGT_K_OTHER, down_convert_kernel, stream_blocks(c, nu), 256, nu, (const double2*)c->Ucb, (float2*)c->Ucb32, 1.0);
        c->ucb32_valid = true;
    }
    float2 *b32 = O32::eo_field(c, 0), *e32 = O32::eo_field(c, 1), *r32 = O32::eo_field(c, 2), *p32 = O32::eo_field(c, 3),
           *u32 = O32::eo_field(c, 4), *t32 = O32::eo_field(c, 5);
    int rc, total = 0, outer = 0, conv = LGT_OK, prev_it = 0;
    double prev_scale = 1.0;
    bool prev_good = false;
    CU(cudaMemsetAsync(x, 0, n * sizeof(double2), c->stream));
    CU(cudaMemcpyAsync(r, b, n * sizeof(double2), cudaMemcpyDeviceToDevice, c->stream));
    if ((rc = O64::redot(c, b, b, c->scal + 3, n)) != LGT_OK) return rc;
    CU(cudaMemcpyAsync(c->h_scal + 3, c->scal + 3, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    const double bb = c->h_scal[3];
    double rr = bb;
    while (bb > 0.0 && rr > tol * tol * bb) {
        if (total >= max_iter || outer >= 40) {
            conv = LGT_ENOCONV;
            break;
        }
        const double scale = 1.0 / sqrt(rr);
        LAUNCH(c, LGT_K_CG_BLAS, down_convert_kernel, nb, 256, n, (const double2*)r, b32, scale);
        double eps = 0.25 * tol * sqrt(bb / rr);
        if (eps < c->inner_tol) eps = c->inner_tol;
        // Reliable update instead of a restart: the last search direction p_k of the previous cycle (the x, p update leaves p alone
        // in the iteration that converges) continues, p = r_true + beta p_k with beta = |r_true|^2 / |r_k|^2, |r_k|^2 = rr / beta_k
        // of the previous cycle's last state; in the units of this cycle (residual scaled to norm 1, p_k rescaled by scale /
        // prev_scale) that is p = r + pcoef p with pcoef = beta_k / (rr_k+1 * (scale / prev_scale)).
        // Only while the true residual is the iterated one to fp32 accuracy (the previous cycle delivered within a factor 10 of
        // what it was asked for): otherwise p_k is not orthogonal to the new residual and CG's step length formula does not hold.
        double pcoef = 0.0;
        if (outer > 0 && prev_it > 0 && prev_good && c->h_st->rr > 0.0 && c->h_st->beta > 0.0)
            pcoef = c->h_st->beta / (c->h_st->rr * (scale / prev_scale));
        int it = 0;
        rc = O32::eo_cg(c, b32, e32, r32, p32, u32, t32, eps, max_iter - total, &it, nullptr, pcoef);
        if (rc != LGT_OK && rc != LGT_ENOCONV) return rc;
        prev_scale = scale;
        prev_it = it;
        total += it;
        outer++;
        LAUNCH(c, LGT_K_CG_BLAS, up_axpy_kernel, nb, 256, n, (double2*)x, (const float2*)e32, 1.0 / scale);
        if ((rc = O64::eo_mhat(c, (const double2*)x, (double2*)u, (double2*)t_o, 0)) != LGT_OK) return rc;
        if ((rc = O64::eo_mhat(c, (const double2*)u, (double2*)q, (double2*)t_o, 1)) != LGT_OK) return rc;
        LAUNCH(c, LGT_K_CG_BLAS, residual_kernel, nb, 256, n, (const double2*)b, (const double2*)q, (double2*)r, c->scal + 3, c->partials, c->counter);
        CU(cudaMemcpyAsync(c->h_scal + 3, c->scal + 3, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        mixed_inner_fallback(c, rr, c->h_scal[3], eps);
        prev_good = c->h_scal[3] <= 100.0 * eps * eps * rr;
        rr = c->h_scal[3];
    }
    c->last_outer = outer;
    if (iters) *iters = total;
    if (conv != LGT_OK) return fail(c, LGT_ENOCONV, "mixed-precision even/odd CG did not reach the tolerance");
    return LGT_OK;
}

// Automatic block swizzle: off while one time slice of links + spinors (48 complex numbers per site) stays well
// inside L2 together with its successor; else the largest divisor Z of Lz whose slab slice does.
// Measured (fp64 Dslash): 48^3 x 96 2347 -> 2030 us, 64^4 3715 -> 3219 us; 32^4 is faster without (191 vs 198 us).
int auto_swizzle(const lgt_ctx* c) {
    const double limit = 28e6;  // bytes of one slab slice
    const double site_bytes = 48.0 * (double)c->esize;
    const long long xy = (long long)c->g.L[0] * c->g.L[1];
    if (xy % 128 != 0) return 0;
    if ((double)xy * c->g.L[2] * site_bytes <= limit) return 0;
    int best = 0;
    for (int Z = 1; Z <= c->g.L[2]; Z++)
        if (c->g.L[2] % Z == 0 && (double)xy * Z * site_bytes <= limit) best = Z;
    return best;
}

// Mixed-precision solve of (D^dag D) x = b on an fp64 handle:
// defect correction x <- x + e, e ~ (D^dag D)^-1 r from a CG run entirely in fp32 (fp32 links, fp32 vectors, the
// same fused kernels instantiated for float) on the residual scaled to unit norm, then r = b - D^dag D x in fp64.
// Stops on the TRUE fp64 residual |r| <= tol |b|.  iters = fp32 CG iterations in total; outer = correction cycles.
// After the loop t = D x (fp64) is what the last residual evaluation left behind, so y = D x costs nothing.
int cg_mixed(lgt_ctx* c, const void* b, void* x, void* y, double tol, int max_iter, int* iters, double* rel) {
    if (c->prec != LGT_F64) return fail(c, LGT_ESTATE, "mixed-precision CG needs an LGT_F64 handle");
    typedef Ops<double> O64;
    typedef Ops<float> O32;
    int rcf = O64::ensure_fermion_links(c);
    if (rcf != LGT_OK) return rcf;
    const size_t n = (size_t)12 * c->g.Vs;
    if (!c->U32) {
        CU(cudaMalloc(&c->U32, (size_t)36 * c->g.Vs * sizeof(float2)));
        for (int i = 0; i < 5; i++) CU(cudaMalloc(&c->ws32[i], n * sizeof(float2)));
        c->u32_valid = false;
    }
    const int nb = stream_blocks(c, n);
    if (!c->u32_valid) {
        const size_t nu = (size_t)36 * c->g.Vs;
        LAUNCH(c, LGT_K_OTHER, down_convert_kernel, stream_blocks(c, nu), 256, nu, (const double2*)c->Uf, (float2*)c->U32, 1.0);
        c->u32_valid = true;
    }
    double2 *r = (double2*)c->ws[1], *q = (double2*)c->ws[2];
    double2* t = (double2*)(y ? y : c->ws[3]);
    float2 *b32 = (float2*)c->ws32[0], *e32 = (float2*)c->ws32[1];
    int rc, total = 0, outer = 0, conv = LGT_OK, prev_it = 0;
    double prev_scale = 1.0;
    bool prev_good = false;
    CU(cudaMemsetAsync(x, 0, n * sizeof(double2), c->stream));
    CU(cudaMemsetAsync(t, 0, n * sizeof(double2), c->stream));
    CU(cudaMemcpyAsync(r, b, n * sizeof(double2), cudaMemcpyDeviceToDevice, c->stream));
    if ((rc = O64::redot(c, b, b, c->scal + 3)) != LGT_OK) return rc;
    CU(cudaMemcpyAsync(c->h_scal + 3, c->scal + 3, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    const double bb = c->h_scal[3];
    double rr = bb;
    while (bb > 0.0 && rr > tol * tol * bb) {
        if (total >= max_iter || outer >= 40) {
            conv = LGT_ENOCONV;
            break;
        }
        const double scale = 1.0 / sqrt(rr);
        LAUNCH(c, LGT_K_CG_BLAS, down_convert_kernel, nb, 256, n, (const double2*)r, b32, scale);
        // the inner solve need not go below what the outer tolerance still asks for
        double eps = 0.25 * tol * sqrt(bb / rr);
        if (eps < c->inner_tol) eps = c->inner_tol;
        // reliable update instead of a restart, as in eo_cg_mixed: p = r + pcoef p_k while the true residual is the iterated one
        double pcoef = 0.0;
        if (outer > 0 && prev_it > 0 && prev_good && c->h_st->rr > 0.0 && c->h_st->beta > 0.0)
            pcoef = c->h_st->beta / (c->h_st->rr * (scale / prev_scale));
        int it = 0;
        rc = O32::cg(c, c->U32, c->ws32[2], c->ws32[3], c->ws32[4], b32, e32, nullptr, eps, max_iter - total, &it, nullptr, pcoef);
        if (rc != LGT_OK && rc != LGT_ENOCONV) return rc;
        prev_scale = scale;
        prev_it = it;
        total += it;
        outer++;
        LAUNCH(c, LGT_K_CG_BLAS, up_axpy_kernel, nb, 256, n, (double2*)x, (const float2*)e32, 1.0 / scale);
        if ((rc = O64::dslash(c, c->Uf, x, t, 0, 0)) != LGT_OK) return rc;
        if ((rc = O64::dslash(c, c->Uf, t, q, 1, 0)) != LGT_OK) return rc;
        LAUNCH(c, LGT_K_CG_BLAS, residual_kernel, nb, 256, n, (const double2*)b, (const double2*)q, r, c->scal + 3, c->partials, c->counter);
        CU(cudaMemcpyAsync(c->h_scal + 3, c->scal + 3, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        prev_good = c->h_scal[3] <= 100.0 * eps * eps * rr;
        rr = c->h_scal[3];
    }
    c->last_outer = outer;
    if (iters) *iters = total;
    if (rel) *rel = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    if (conv != LGT_OK) return fail(c, LGT_ENOCONV, "mixed-precision CG did not reach the tolerance");
    return LGT_OK;
}

// X = ws[0], Y = ws[3] (full native fields, as the fused force kernel takes them) for the handle's fermion action and
// solver; dev_SF (may be null) receives S_F on the device.  y == false: only X (and S_F) are wanted.
//   LGT_ACTION_FULL: X = (D^dag D)^-1 phi, Y = D X, S_F = Re <phi, X>   (plain or mixed-precision CG)
//   LGT_ACTION_EO:   X_e = (M^dag M)^-1 phi_e, ...  (Ops::eo_solve_xy), S_F = Re <phi_e, X_e>
int solve(lgt_ctx* c, bool y, double tol, int max_iter, int* iters, double* dev_SF) {
    int rc, conv;
    if (c->action == LGT_ACTION_EO)
        return DISPATCH(c, eo_solve_xy, c, y ? c->ws[0] : nullptr, y ? c->ws[3] : nullptr, tol, max_iter, iters, dev_SF);
    void* Y = y ? c->ws[3] : nullptr;
    if ((rc = DISPATCH(c, ensure_fermion_links, c)) != LGT_OK) return rc;
    if (c->solver == LGT_SOLVER_MIXED_CG && c->prec == LGT_F64)
        conv = cg_mixed(c, c->phi, c->ws[0], Y, tol, max_iter, iters, nullptr);
    else
        conv = DISPATCH(c, cg, c, c->Uf, c->ws[1], c->ws[2], c->ws[3], c->phi, c->ws[0], Y, tol, max_iter, iters, nullptr);
    if (conv != LGT_OK && conv != LGT_ENOCONV) return conv;
    if (dev_SF && (rc = DISPATCH(c, redot, c, c->phi, c->ws[0], dev_SF, 0)) != LGT_OK) return rc;
    return conv;
}

bool fermions_on(const lgt_ctx* c) { return c->kappa != 0.0 && c->has_phi; }

// Metropolis uniform: Philox4x32-10 at counter (0, 0, stream 3, trajectory), first uniform (reading A-25)
double metropolis_uniform(unsigned long long seed, unsigned traj) {
    unsigned c[4] = {0u, 0u, 3u, traj};
    unsigned k0 = (unsigned)(seed & 0xffffffffull), k1 = (unsigned)(seed >> 32);
    for (int round = 0; round < 10; round++) {
        const unsigned long long p0 = 0xD2511F53ull * c[0], p1 = 0xCD9E8D57ull * c[2];
        const unsigned n0 = (unsigned)(p1 >> 32) ^ c[1] ^ k0, n2 = (unsigned)(p0 >> 32) ^ c[3] ^ k1;
        c[0] = n0;
        c[1] = (unsigned)p1;
        c[2] = n2;
        c[3] = (unsigned)p0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    const unsigned long long a = ((unsigned long long)c[1] << 32) | c[0];
    return ((double)(a >> 11) + 0.5) * 0x1p-53;
}

// Pi -= eps F^g
int kick_gauge(lgt_ctx* c, double eps) {
    p_ready(c);
    p_ready(c);
    return DISPATCH(c, gauge_force, c, c->P, 1, eps);
}
// Pi -= eps F^f (solve, then the fused force kernel); nothing if there are no fermions
int kick_fermion(lgt_ctx* c, double eps, double tol, int max_iter, int* cg_iters) {
    int rc, it = 0, conv = LGT_OK;
    if (fermions_on(c)) {
        rc = solve(c, true, tol, max_iter, &it, nullptr);
        if (rc == LGT_ENOCONV) conv = rc;
        else if (rc != LGT_OK) return rc;
        p_ready(c);
        if ((rc = DISPATCH(c, fermion_force, c, c->ws[0], c->ws[3], c->P, 1, eps)) != LGT_OK) return rc;
    }
    if (cg_iters) *cg_iters = it;
    return conv;
}
// Pi -= eps (F^g + F^f).  The solve comes first: it does not touch Pi, so a pending asynchronous upload of the momenta
// (lgt_set_momenta_host_async) overlaps it; the two force kernels then update Pi in the same order as before
// (gauge, then fermion), so the result is bitwise unchanged.
int kick(lgt_ctx* c, double eps, double tol, int max_iter, int* cg_iters) {
    int rc, it = 0, conv = LGT_OK;
    const bool ferm = fermions_on(c);
    if (ferm) {
        rc = solve(c, true, tol, max_iter, &it, nullptr);
        if (rc == LGT_ENOCONV) conv = rc;
        else if (rc != LGT_OK) return rc;
    }
    if ((rc = kick_gauge(c, eps)) != LGT_OK) return rc;
    if (ferm && (rc = DISPATCH(c, fermion_force, c, c->ws[0], c->ws[3], c->P, 1, eps)) != LGT_OK) return rc;
    if (cg_iters) *cg_iters = it;
    return conv;
}

// MD trajectory of nsteps steps of size dt, adjacent kicks merged (include/lgt.h "lgt_set_integrator").  S supplies the
// moves: kick(eps, &it) with both forces, kick_gauge(eps), kick_fermion(eps, &it), drift(eps) -- one handle, or all slabs
// of a decomposed lattice in lockstep.
// The gauge part of one Sexton-Weingarten step: m leapfrog steps of size h with the gauge force alone
template <class S> int plain_inner_gauge_steps(S& s, double h, int m) {
    int rc;
    if ((rc = s.kick_gauge(0.5 * h)) != LGT_OK) return rc;
    for (int i = 0; i < m; i++) {
        if ((rc = s.drift(h)) != LGT_OK) return rc;
        if ((rc = s.kick_gauge((i == m - 1) ? 0.5 * h : h)) != LGT_OK) return rc;
    }
    return LGT_OK;
}
template <class S> int integrate_with(S& s, int integrator, int n_inner, int nsteps, double dt, long* cg_iters) {
    int rc, it = 0, conv = LGT_OK;
    long total = 0;
#define STEP(call)                           \
    do {                                     \
        it = 0;                              \
        rc = (call);                         \
        if (rc == LGT_ENOCONV) conv = rc;    \
        else if (rc != LGT_OK) return rc;    \
        total += it;                         \
    } while (0)
    if (nsteps > 0 && integrator == LGT_INT_LEAPFROG) {
        STEP(s.kick(0.5 * dt, &it));
        for (int n = 0; n < nsteps; n++) {
            STEP(s.drift(dt));
            STEP(s.kick((n == nsteps - 1) ? 0.5 * dt : dt, &it));
        }
    } else if (nsteps > 0 && integrator == LGT_INT_OMELYAN) {
        const double lam = 0.1931833275037836;
        STEP(s.kick(lam * dt, &it));
        for (int n = 0; n < nsteps; n++) {
            STEP(s.drift(0.5 * dt));
            STEP(s.kick((1.0 - 2.0 * lam) * dt, &it));
            STEP(s.drift(0.5 * dt));
            STEP(s.kick((n == nsteps - 1) ? lam * dt : 2.0 * lam * dt, &it));
        }
    } else if (nsteps > 0) {  // Sexton-Weingarten: fermion force outside, m gauge leapfrog steps inside
        const int m = n_inner;
        const double h = dt / m;
        STEP(s.kick_fermion(0.5 * dt, &it));
        for (int n = 0; n < nsteps; n++) {
            STEP(s.inner_gauge_steps(h, m));
            STEP(s.kick_fermion((n == nsteps - 1) ? 0.5 * dt : dt, &it));
        }
    }
#undef STEP
    if (cg_iters) *cg_iters = total;
    return conv;
}
struct HandleMoves {
    lgt_ctx* c;
    double tol;
    int max_iter;
    int kick(double eps, int* it) { return ::kick(c, eps, tol, max_iter, it); }
    int kick_gauge(double eps) { return ::kick_gauge(c, eps); }
    int kick_fermion(double eps, int* it) { return ::kick_fermion(c, eps, tol, max_iter, it); }
    int drift(double eps) { return DISPATCH(c, link_update, c, eps); }
    // The 2 m + 1 launches of the inner gauge loop have the same arguments in every outer step of a trajectory (and in
    // every trajectory with the same dt and m), and on the paper's lattice sizes (6^4 - 16^4) each is a
    // few microseconds of work: they are captured once as a CUDA graph and replayed with one launch, like the CG chunks.
    int inner_gauge_steps(double h, int m) {
        unsigned long long hbits;
        memcpy(&hbits, &h, sizeof hbits);
        const void* const key[7] = {c->U, c->P, (const void*)hbits, (const void*)(size_t)m,
                                    (const void*)(size_t)c->variant[LGT_K_GAUGE_FORCE], nullptr, (const void*)c->esize};
        HandleMoves& self = *this;
        const int rc = chunk_graph(c, 2, key, [&]() -> int { return plain_inner_gauge_steps(self, h, m); });
        invalidate_link_copies(c);  // the replayed link updates changed U behind the host-side flags
        return rc;
    }
};
int integrate(lgt_ctx* c, int nsteps, double dt, double tol, int max_iter, long* cg_iters) {
    HandleMoves m{c, tol, max_iter};
    return integrate_with(m, c->integrator, c->n_inner, nsteps, dt, cg_iters);
}

int hamiltonian(lgt_ctx* c, double tol, int max_iter, double* S_g, double* S_F, double* K, int* cg_iters) {
    int rc, it = 0, conv = LGT_OK;
    if ((rc = DISPATCH(c, plaquette_sum, c, c->scal + 0)) != LGT_OK) return rc;
    if ((rc = DISPATCH(c, kinetic, c, c->scal + 1)) != LGT_OK) return rc;
    bool ferm = fermions_on(c) && S_F != nullptr;
    if (ferm) {
        rc = solve(c, false, tol, max_iter, &it, c->scal + 2);
        if (rc == LGT_ENOCONV) conv = rc;
        else if (rc != LGT_OK) return rc;
    }
    if ((rc = read_scalars(c, 3)) != LGT_OK) return rc;
    if (S_g) *S_g = c->beta * (6.0 * (double)c->g.V - c->h_scal[0]);
    if (K) *K = c->h_scal[1];
    if (S_F) *S_F = ferm ? c->h_scal[2] : 0.0;
    if (cg_iters) *cg_iters = it;
    return conv;
}

}  // namespace

namespace {
int eo_check(lgt_ctx* c, const char* what) {
    for (int m = 0; m < 4; m++)
        if (c->g.L[m] % 2) return fail(c, LGT_EINVAL, what);
    return LGT_OK;
}
template <class T> int eo_mhat_canonical(lgt_ctx* c, const void* in, void* out, int dagger) {
    typedef Ops<T> O;
    int rc;
    if ((rc = O::eo_ensure(c)) != LGT_OK) return rc;
    if ((rc = O::to_native(c, in, c->ws[5], 12)) != LGT_OK) return rc;
    if ((rc = O::eo_split(c, c->ws[5], O::eo_field(c, 4))) != LGT_OK) return rc;          // fields 4, 5 = (in_e, in_o)
    if ((rc = O::eo_mhat(c, O::eo_field(c, 4), O::eo_field(c, 2), O::eo_field(c, 7), dagger)) != LGT_OK) return rc;
    CU(cudaMemsetAsync(O::eo_field(c, 3), 0, (size_t)12 * c->g.Vhs * sizeof(typename O::T2), c->stream));  // odd part of out = 0
    if ((rc = O::eo_merge(c, O::eo_field(c, 2), c->ws[5])) != LGT_OK) return rc;
    return O::from_native(c, c->ws[5], out, 12);
}
template <class T> int eo_cg_canonical(lgt_ctx* c, const void* b, void* x, double tol, int max_iter, int* iters, double* rel) {
    typedef Ops<T> O;
    int rc;
    if ((rc = O::eo_ensure(c)) != LGT_OK) return rc;
    if ((rc = O::to_native(c, b, c->ws[5], 12)) != LGT_OK) return rc;
    if ((rc = O::eo_split(c, c->ws[5], O::eo_field(c, 4))) != LGT_OK) return rc;
    int conv = O::eo_cg(c, O::eo_field(c, 4), O::eo_field(c, 0), O::eo_field(c, 5), O::eo_field(c, 6), O::eo_field(c, 2),
                        O::eo_field(c, 7), tol, max_iter, iters, rel);
    if (conv != LGT_OK && conv != LGT_ENOCONV) return conv;
    CU(cudaMemsetAsync(O::eo_field(c, 1), 0, (size_t)12 * c->g.Vhs * sizeof(typename O::T2), c->stream));  // odd part of x = 0
    if ((rc = O::eo_merge(c, O::eo_field(c, 0), c->ws[5])) != LGT_OK) return rc;
    if ((rc = O::from_native(c, c->ws[5], x, 12)) != LGT_OK) return rc;
    return conv;
}
}  // namespace

#define CHECK_CTX(c) \
    if (!(c)) return LGT_EINVAL; \
    DeviceGuard guard_((c)->device)
// calls that need neighbours or global sums are wrong on one time slab of a decomposed lattice: use lgt_dd_*
#define NOT_SLAB(c) \
    if ((c)->dd_links_valid) return fail((c), LGT_ESTATE, "this handle is a time slab of a decomposed lattice: use the lgt_dd_* call")

extern "C" {

const char* lgt_version(void) { return "lgt-b200 0.2 (sm_100a)"; }

const char* lgt_last_error(const lgt_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int lgt_create(lgt_ctx** out, const int dims[4], double beta, double kappa, const int bc[4], int precision, int device,
               void* cuda_stream) {
    lgt_ctx* c = nullptr;
    if (!out || !dims || !bc) return fail(nullptr, LGT_EINVAL, "lgt_create: null argument");
    *out = nullptr;
    long long V = 1;
    for (int m = 0; m < 4; m++) {
        if (dims[m] < 1) return fail(nullptr, LGT_EINVAL, "lgt_create: dims must be >= 1");
        if (bc[m] != 1 && bc[m] != -1) return fail(nullptr, LGT_EINVAL, "lgt_create: bc entries must be +1 or -1");
        V *= dims[m];
        if (V > (1LL << 30)) return fail(nullptr, LGT_EINVAL, "lgt_create: lattice too large for 32-bit site indices");
    }
    if (precision != LGT_F64 && precision != LGT_F32) return fail(nullptr, LGT_EINVAL, "lgt_create: bad precision");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, LGT_ECUDA, "lgt_create: no CUDA device (there is no CPU fallback)", e);
    if (device < 0 || device >= ndev) return fail(nullptr, LGT_EINVAL, "lgt_create: bad device index");
    try {
        c = new lgt_ctx();
    } catch (const std::bad_alloc&) {
        return fail(nullptr, LGT_ENOMEM, "lgt_create: host allocation failed");
    }
    DeviceGuard guard(device);
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->beta = beta;
    c->kappa = kappa;
    c->prec = precision;
    c->esize = precision == LGT_F64 ? 16 : 8;
    int stride = 1;
    for (int m = 0; m < 4; m++) {
        c->g.L[m] = dims[m];
        c->g.bc[m] = bc[m];
        c->g.stride[m] = stride;
        stride *= dims[m];
    }
    c->g.V = (int)V;
    c->g.Vs = (int)((V + 31) / 32 * 32);
    c->g.Vh = (int)(V / 2);
    c->g.Vhs = (c->g.Vh + 31) / 32 * 32;
    c->g.swz_cxy = (int)(((long long)dims[0] * dims[1]) / 128);
    c->g.swz_Z = auto_swizzle(c);
    c->g.s_begin = 0;
    c->g.s_end = c->g.V;
    c->g.t_off = 0;
    c->g.Lt_glob = c->g.L[3];
    c->g.site_off = 0;
    c->g.z_lo = 0;
    c->g.z_hi = c->g.L[2];
    c->g.z_off = 0;
    c->g.Lz_glob = c->g.L[2];
    c->g.h_begin = 0;
    c->g.h_end = c->g.Vh;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    c->red_blocks = sms * 8;
    c->num_sms = sms;
    int rc = LGT_OK;
    auto alloc = [&](void** p, size_t bytes) {
        if (rc != LGT_OK) return;
        cudaError_t ee = cudaMalloc(p, bytes);
        if (ee != cudaSuccess) rc = fail(nullptr, ee == cudaErrorMemoryAllocation ? LGT_ENOMEM : LGT_ECUDA, "lgt_create: cudaMalloc", ee);
    };
    alloc(&c->U, links_bytes(c));
    alloc(&c->P, mom_bytes(c));
    alloc(&c->phi, spinor_bytes(c));
    for (int i = 0; i < 6; i++) alloc(&c->ws[i], spinor_bytes(c));
    size_t npart = (size_t)(c->g.Vs / 32) + c->red_blocks + 64;
    alloc((void**)&c->partials, npart * sizeof(double));
    alloc((void**)&c->counter, sizeof(unsigned));
    alloc((void**)&c->st, sizeof(CgState));
    alloc((void**)&c->st2, sizeof(CgState));
    alloc((void**)&c->scal, 8 * sizeof(double));
    if (rc == LGT_OK && (cudaMallocHost((void**)&c->h_st, sizeof(CgState)) != cudaSuccess ||
                         cudaMallocHost((void**)&c->h_scal, 8 * sizeof(double)) != cudaSuccess))
        rc = fail(nullptr, LGT_ENOMEM, "lgt_create: cudaMallocHost failed");
    if (rc == LGT_OK) {
        bool ok = cudaMemsetAsync(c->counter, 0, sizeof(unsigned), c->stream) == cudaSuccess &&
                  cudaMemsetAsync(c->st, 0, sizeof(CgState), c->stream) == cudaSuccess &&
                  cudaMemsetAsync(c->P, 0, mom_bytes(c), c->stream) == cudaSuccess &&
                  cudaMemsetAsync(c->phi, 0, spinor_bytes(c), c->stream) == cudaSuccess;
        for (int i = 0; i < 6 && ok; i++) ok = cudaMemsetAsync(c->ws[i], 0, spinor_bytes(c), c->stream) == cudaSuccess;
        if (!ok) rc = fail(nullptr, LGT_ECUDA, "lgt_create: cudaMemsetAsync failed");
    }
    if (rc == LGT_OK) {
        rc = DISPATCH(c, unit_links, c);
        if (rc != LGT_OK) g_create_error = c->err;
    }
    if (rc == LGT_OK && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = fail(nullptr, LGT_ECUDA, "lgt_create: sync failed");
    if (rc != LGT_OK) {
        lgt_destroy(c);
        return rc;
    }
    *out = c;
    return LGT_OK;
}

int lgt_destroy(lgt_ctx* c) {
    if (!c) return LGT_OK;
    DeviceGuard guard(c->device);
    cudaStreamSynchronize(c->stream);
    if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);  // pending asynchronous host transfers
    cudaFree(c->U);
    cudaFree(c->P);
    cudaFree(c->phi);
    for (int i = 0; i < 6; i++) cudaFree(c->ws[i]);
    cudaFree(c->F);
    cudaFree(c->U32);
    cudaFree(c->Ucb);
    cudaFree(c->Usave);
    for (int i = 0; i < LGT_MAX_SMEAR; i++) {
        cudaFree(c->Usm[i]);
        cudaFree(c->Asm[i]);
    }
    cudaFree(c->F2);
    cudaFree(c->F3);
    cudaFree(c->F4);
    cudaFree(c->eo);
    cudaFree(c->Ucb32);
    cudaFree(c->eo32);
    for (int i = 0; i < 5; i++) cudaFree(c->ws32[i]);
    cudaFree(c->stage);
    cudaFree(c->stage_p_in);
    cudaFree(c->stage_u_out);
    cudaFree(c->stage_p_out);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (cudaEvent_t e : {c->ev_main, c->ev_p_up, c->ev_u_down, c->ev_p_down})
        if (e) cudaEventDestroy(e);
    cudaFree(c->partials);
    cudaFree(c->counter);
    cudaFree(c->coop_counter);
    cudaFree(c->st);
    cudaFree(c->st2);
    cudaFree(c->scal);
    if (c->h_st) cudaFreeHost(c->h_st);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    for (const lgt_ctx::ChunkGraph& g : c->graphs) cudaGraphExecDestroy(g.exec);
    if (c->capture_stream) cudaStreamDestroy(c->capture_stream);
    delete c;
    return LGT_OK;
}

int lgt_timing_enable(lgt_ctx* c, int enable) {
    CHECK_CTX(c);
    c->timing = enable != 0;
    return LGT_OK;
}
int lgt_timing_reset(lgt_ctx* c) {
    CHECK_CTX(c);
    CU(cudaStreamSynchronize(c->stream));
    c->ev_used = 0;
    c->ev_class.clear();
    return LGT_OK;
}
int lgt_timing_read(lgt_ctx* c, int kernel_class, double* ms_total, long* launches) {
    CHECK_CTX(c);
    if (kernel_class < 0 || kernel_class >= LGT_K_COUNT) return fail(c, LGT_EINVAL, "lgt_timing_read: bad kernel class");
    CU(cudaStreamSynchronize(c->stream));
    double total = 0.0;
    long n = 0;
    for (size_t i = 0; i < c->ev_class.size(); i++) {
        if (c->ev_class[i] != kernel_class) continue;
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, c->ev_pool[2 * i], c->ev_pool[2 * i + 1]));
        total += ms;
        n++;
    }
    if (ms_total) *ms_total = total;
    if (launches) *launches = n;
    return LGT_OK;
}

long lgt_launch_count(const lgt_ctx* c) { return c ? c->launches : 0; }
int lgt_set_block_swizzle(lgt_ctx* c, int z_planes, int* in_effect) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (z_planes < 0) {
        c->g.swz_Z = auto_swizzle(c);
    } else if (z_planes == 0) {
        c->g.swz_Z = 0;
    } else {
        if (c->g.L[2] % z_planes != 0 || ((long long)c->g.L[0] * c->g.L[1]) % 128 != 0)
            return fail(c, LGT_EINVAL, "lgt_set_block_swizzle: Z must divide Lz and Lx*Ly must be a multiple of 128");
        c->g.swz_Z = z_planes;
    }
    if (in_effect) *in_effect = c->g.swz_Z;
    return LGT_OK;
}
int lgt_set_kernel_variant(lgt_ctx* c, int kernel_class, int variant, int* in_effect) {
    CHECK_CTX(c);
    if (kernel_class < 0 || kernel_class >= LGT_K_COUNT) return fail(c, LGT_EINVAL, "lgt_set_kernel_variant: unknown kernel class");
    if (variant >= 0) {
        const int nvar = (kernel_class == LGT_K_DSLASH) ? 13 : (kernel_class == LGT_K_GAUGE_FORCE) ? 4 : (kernel_class == LGT_K_CG_BLAS) ? 4 : 1;
        if (variant >= nvar) return fail(c, LGT_EINVAL, "lgt_set_kernel_variant: this kernel class has no such variant");
        if (c->variant[kernel_class] != variant) {
            // captured CG chunks hold the old kernels
            for (lgt_ctx::ChunkGraph& g : c->graphs) cudaGraphExecDestroy(g.exec);
            c->graphs.clear();
        }
        c->variant[kernel_class] = variant;
    }
    if (in_effect) *in_effect = c->variant[kernel_class];
    return LGT_OK;
}
void* lgt_stream(const lgt_ctx* c) { return c ? (void*)c->stream : nullptr; }
long lgt_native_spinor_bytes(const lgt_ctx* c) { return c ? (long)spinor_bytes(c) : 0; }

// ---- state
int lgt_set_links(lgt_ctx* c, const void* U) {
    CHECK_CTX(c);
    if (!U) return fail(c, LGT_EINVAL, "lgt_set_links: null pointer");
    c->u32_valid = false;
    c->usm_valid = false;
    if (c->dd_links_valid) *c->dd_links_valid = false;
    c->ucb_valid = false;
    c->ucb32_valid = false;
    c->inner_exact = false;
    return DISPATCH(c, to_native, c, U, c->U, 36);
}
int lgt_get_links(lgt_ctx* c, void* U) {
    CHECK_CTX(c);
    if (!U) return fail(c, LGT_EINVAL, "lgt_get_links: null pointer");
    return DISPATCH(c, from_native, c, c->U, U, 36);
}
int lgt_set_momenta(lgt_ctx* c, const void* P) {
    CHECK_CTX(c);
    if (!P) return fail(c, LGT_EINVAL, "lgt_set_momenta: null pointer");
    p_ready(c);
    return DISPATCH(c, momenta_to_native, c, P, c->P);
}
int lgt_get_momenta(lgt_ctx* c, void* P) {
    CHECK_CTX(c);
    if (!P) return fail(c, LGT_EINVAL, "lgt_get_momenta: null pointer");
    p_ready(c);
    return DISPATCH(c, momenta_from_native, c, c->P, P);
}
int lgt_set_pseudofermion(lgt_ctx* c, const void* phi) {
    CHECK_CTX(c);
    if (!phi) return fail(c, LGT_EINVAL, "lgt_set_pseudofermion: null pointer");
    int rc = DISPATCH(c, to_native, c, phi, c->phi, 12);
    if (rc == LGT_OK) c->has_phi = true;
    return rc;
}

#define HOST_SET(name, devcall, bytes_expr)                                                         \
    int name(lgt_ctx* c, const void* h) {                                                           \
        CHECK_CTX(c);                                                                               \
        if (!h) return fail(c, LGT_EINVAL, #name ": null pointer");                                 \
        size_t bytes = (bytes_expr);                                                                \
        int rc = ensure_stage(c, bytes);                                                            \
        if (rc != LGT_OK) return rc;                                                                \
        CU(cudaMemcpyAsync(c->stage, h, bytes, cudaMemcpyHostToDevice, c->stream));                 \
        rc = devcall(c, c->stage);                                                                  \
        if (rc != LGT_OK) return rc;                                                                \
        CU(cudaStreamSynchronize(c->stream));                                                       \
        return LGT_OK;                                                                              \
    }
#define HOST_GET(name, devcall, bytes_expr)                                                         \
    int name(lgt_ctx* c, void* h) {                                                                 \
        CHECK_CTX(c);                                                                               \
        if (!h) return fail(c, LGT_EINVAL, #name ": null pointer");                                 \
        size_t bytes = (bytes_expr);                                                                \
        int rc = ensure_stage(c, bytes);                                                            \
        if (rc != LGT_OK) return rc;                                                                \
        rc = devcall(c, c->stage);                                                                  \
        if (rc != LGT_OK) return rc;                                                                \
        CU(cudaMemcpyAsync(h, c->stage, bytes, cudaMemcpyDeviceToHost, c->stream));                 \
        CU(cudaStreamSynchronize(c->stream));                                                       \
        return LGT_OK;                                                                              \
    }
HOST_SET(lgt_set_links_host, lgt_set_links, (size_t)36 * (c->g.s_end - c->g.s_begin) * c->esize)
HOST_GET(lgt_get_links_host, lgt_get_links, (size_t)36 * (c->g.s_end - c->g.s_begin) * c->esize)
HOST_SET(lgt_set_momenta_host, lgt_set_momenta, (size_t)36 * (c->g.s_end - c->g.s_begin) * c->esize)
HOST_GET(lgt_get_momenta_host, lgt_get_momenta, (size_t)36 * (c->g.s_end - c->g.s_begin) * c->esize)
HOST_SET(lgt_set_pseudofermion_host, lgt_set_pseudofermion, (size_t)12 * (c->g.s_end - c->g.s_begin) * c->esize)

// ---- asynchronous host transfers
namespace {
int ensure_async(lgt_ctx* c) {
    if (c->dd_links_valid) return fail(c, LGT_ESTATE, "the asynchronous host transfers are for undivided lattices");
    if (c->copy_stream) return LGT_OK;
    CU(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&c->ev_main, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&c->ev_p_up, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&c->ev_u_down, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&c->ev_p_down, cudaEventDisableTiming));
    return LGT_OK;
}
// device -> host of one field: conversion on the handle's stream into the field's own staging buffer (after the previous
// download from that buffer has left it), then the copy on the copy stream
int download_async(lgt_ctx* c, void** stage, bool* pending, cudaEvent_t done, int (*convert)(lgt_ctx*, void*), void* h, size_t bytes) {
    int rc;
    if ((rc = ensure_async(c)) != LGT_OK) return rc;
    if (!*stage) CU(cudaMalloc(stage, bytes));
    if (*pending) CU(cudaStreamWaitEvent(c->stream, done, 0));
    if ((rc = convert(c, *stage)) != LGT_OK) return rc;
    CU(cudaEventRecord(c->ev_main, c->stream));
    CU(cudaStreamWaitEvent(c->copy_stream, c->ev_main, 0));
    CU(cudaMemcpyAsync(h, *stage, bytes, cudaMemcpyDeviceToHost, c->copy_stream));
    CU(cudaEventRecord(done, c->copy_stream));
    *pending = true;
    return LGT_OK;
}
}  // namespace

int lgt_set_momenta_host_async(lgt_ctx* c, const void* h) {
    CHECK_CTX(c);
    if (!h) return fail(c, LGT_EINVAL, "lgt_set_momenta_host_async: null pointer");
    int rc;
    if ((rc = ensure_async(c)) != LGT_OK) return rc;
    const size_t bytes = (size_t)36 * c->g.V * c->esize;
    if (!c->stage_p_in) CU(cudaMalloc(&c->stage_p_in, bytes));
    p_ready(c);  // an earlier pending upload: keep the order
    // everything enqueued so far may still read or write Pi (and the staging buffer): the copy stream starts after it
    CU(cudaEventRecord(c->ev_main, c->stream));
    CU(cudaStreamWaitEvent(c->copy_stream, c->ev_main, 0));
    CU(cudaMemcpyAsync(c->stage_p_in, h, bytes, cudaMemcpyHostToDevice, c->copy_stream));
    cudaStream_t const main_stream = c->stream;
    c->stream = c->copy_stream;  // the conversion kernel follows the copy on the copy stream
    rc = DISPATCH(c, momenta_to_native, c, c->stage_p_in, c->P);
    c->stream = main_stream;
    if (rc != LGT_OK) return rc;
    CU(cudaEventRecord(c->ev_p_up, c->copy_stream));
    c->p_pending = true;
    return LGT_OK;
}
int lgt_get_links_host_async(lgt_ctx* c, void* h) {
    CHECK_CTX(c);
    if (!h) return fail(c, LGT_EINVAL, "lgt_get_links_host_async: null pointer");
    return download_async(c, &c->stage_u_out, &c->u_down_pending, c->ev_u_down, [](lgt_ctx* cc, void* st) { return lgt_get_links(cc, st); }, h,
                          (size_t)36 * c->g.V * c->esize);
}
int lgt_get_momenta_host_async(lgt_ctx* c, void* h) {
    CHECK_CTX(c);
    if (!h) return fail(c, LGT_EINVAL, "lgt_get_momenta_host_async: null pointer");
    return download_async(c, &c->stage_p_out, &c->p_down_pending, c->ev_p_down, [](lgt_ctx* cc, void* st) { return lgt_get_momenta(cc, st); }, h,
                          (size_t)36 * c->g.V * c->esize);
}
int lgt_host_transfers_wait(lgt_ctx* c) {
    CHECK_CTX(c);
    if (c->copy_stream) CU(cudaStreamSynchronize(c->copy_stream));
    c->u_down_pending = c->p_down_pending = false;
    return LGT_OK;
}

// ---- actions
int lgt_action(lgt_ctx* c, double tol, int max_iter, double* S_g, double* S_F, double* K, int* cg_iters) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    return hamiltonian(c, tol, max_iter, S_g, S_F, K, cg_iters);
}
int lgt_plaquette(lgt_ctx* c, double* plaq) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!plaq) return fail(c, LGT_EINVAL, "lgt_plaquette: null pointer");
    int rc = DISPATCH(c, plaquette_sum, c, c->scal + 0);
    if (rc != LGT_OK) return rc;
    if ((rc = read_scalars(c, 1)) != LGT_OK) return rc;
    *plaq = c->h_scal[0] / (6.0 * (double)c->g.V);
    return LGT_OK;
}

// ---- Dirac operator
int lgt_spinor_to_native(lgt_ctx* c, const void* canonical, void* native) {
    CHECK_CTX(c);
    if (!canonical || !native || canonical == native) return fail(c, LGT_EINVAL, "lgt_spinor_to_native: bad pointers");
    return DISPATCH(c, to_native, c, canonical, native, 12);
}
int lgt_spinor_from_native(lgt_ctx* c, const void* native, void* canonical) {
    CHECK_CTX(c);
    if (!canonical || !native || canonical == native) return fail(c, LGT_EINVAL, "lgt_spinor_from_native: bad pointers");
    return DISPATCH(c, from_native, c, native, canonical, 12);
}
int lgt_dslash_native(lgt_ctx* c, const void* in, void* out, int dagger) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!in || !out || in == out) return fail(c, LGT_EINVAL, "lgt_dslash_native: in and out must be distinct non-null buffers");
    int rcf = DISPATCH(c, ensure_fermion_links, c);
    if (rcf != LGT_OK) return rcf;
    return DISPATCH(c, dslash, c, c->Uf, in, out, dagger ? 1 : 0, 0);
}
int lgt_dslash(lgt_ctx* c, const void* in, void* out, int dagger) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!in || !out || in == out) return fail(c, LGT_EINVAL, "lgt_dslash: in and out must be distinct non-null buffers");
    int rc;
    if ((rc = DISPATCH(c, ensure_fermion_links, c)) != LGT_OK) return rc;
    if ((rc = DISPATCH(c, to_native, c, in, c->ws[3], 12)) != LGT_OK) return rc;
    if ((rc = DISPATCH(c, dslash, c, c->Uf, c->ws[3], c->ws[4], dagger ? 1 : 0, 0)) != LGT_OK) return rc;
    return DISPATCH(c, from_native, c, c->ws[4], out, 12);
}

// ---- solver
int lgt_cg_native(lgt_ctx* c, const void* b, void* x, void* y, double tol, int max_iter, int* iters, double* rel_resid) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!b || !x || b == x) return fail(c, LGT_EINVAL, "lgt_cg_native: bad pointers");
    if (!(tol >= 0.0) || max_iter < 0) return fail(c, LGT_EINVAL, "lgt_cg_native: bad tol / max_iter");
    int rcf = DISPATCH(c, ensure_fermion_links, c);
    if (rcf != LGT_OK) return rcf;
    return DISPATCH(c, cg, c, c->Uf, c->ws[1], c->ws[2], c->ws[3], b, x, y, tol, max_iter, iters, rel_resid);
}
int lgt_cg(lgt_ctx* c, const void* b, void* x, double tol, int max_iter, int* iters, double* rel_resid) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!b || !x) return fail(c, LGT_EINVAL, "lgt_cg: null pointer");
    if (!(tol >= 0.0) || max_iter < 0) return fail(c, LGT_EINVAL, "lgt_cg: bad tol / max_iter");
    int rc;
    if ((rc = DISPATCH(c, ensure_fermion_links, c)) != LGT_OK) return rc;
    if ((rc = DISPATCH(c, to_native, c, b, c->ws[5], 12)) != LGT_OK) return rc;
    int conv = DISPATCH(c, cg, c, c->Uf, c->ws[1], c->ws[2], c->ws[3], c->ws[5], c->ws[0], nullptr, tol, max_iter, iters, rel_resid);
    if (conv != LGT_OK && conv != LGT_ENOCONV) return conv;
    if ((rc = DISPATCH(c, from_native, c, c->ws[0], x, 12)) != LGT_OK) return rc;
    return conv;
}

int lgt_set_fermion_action(lgt_ctx* c, int action) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (action != LGT_ACTION_FULL && action != LGT_ACTION_EO) return fail(c, LGT_EINVAL, "lgt_set_fermion_action: unknown action");
    if (action == LGT_ACTION_EO)
        for (int m = 0; m < 4; m++)
            if (c->g.L[m] % 2) return fail(c, LGT_EINVAL, "lgt_set_fermion_action: the even/odd action needs every extent even");
    c->action = action;
    return LGT_OK;
}
int lgt_eo_mhat(lgt_ctx* c, const void* in, void* out, int dagger) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!in || !out || in == out) return fail(c, LGT_EINVAL, "lgt_eo_mhat: in and out must be distinct non-null buffers");
    int rc = eo_check(c, "lgt_eo_mhat: every extent must be even");
    if (rc != LGT_OK) return rc;
    return c->prec == LGT_F64 ? eo_mhat_canonical<double>(c, in, out, dagger ? 1 : 0) : eo_mhat_canonical<float>(c, in, out, dagger ? 1 : 0);
}
int lgt_eo_cg(lgt_ctx* c, const void* b, void* x, double tol, int max_iter, int* iters, double* rel_resid) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!b || !x) return fail(c, LGT_EINVAL, "lgt_eo_cg: null pointer");
    if (!(tol >= 0.0) || max_iter < 0) return fail(c, LGT_EINVAL, "lgt_eo_cg: bad tol / max_iter");
    int rc = eo_check(c, "lgt_eo_cg: every extent must be even");
    if (rc != LGT_OK) return rc;
    return c->prec == LGT_F64 ? eo_cg_canonical<double>(c, b, x, tol, max_iter, iters, rel_resid)
                              : eo_cg_canonical<float>(c, b, x, tol, max_iter, iters, rel_resid);
}

int lgt_set_solver(lgt_ctx* c, int solver, double inner_tol) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (solver != LGT_SOLVER_CG && solver != LGT_SOLVER_MIXED_CG) return fail(c, LGT_EINVAL, "lgt_set_solver: unknown solver");
    if (solver == LGT_SOLVER_MIXED_CG && c->prec != LGT_F64) return fail(c, LGT_EINVAL, "lgt_set_solver: mixed precision needs an LGT_F64 handle");
    if (solver == LGT_SOLVER_MIXED_CG && !(inner_tol > 0.0 && inner_tol < 1.0)) return fail(c, LGT_EINVAL, "lgt_set_solver: inner_tol must be in (0, 1)");
    c->solver = solver;
    if (solver == LGT_SOLVER_MIXED_CG) c->inner_tol = inner_tol;
    return LGT_OK;
}
int lgt_cg_mixed(lgt_ctx* c, const void* b, void* x, double tol, int max_iter, double inner_tol, int* inner_iters, int* outer_cycles,
                 double* rel_resid) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!b || !x) return fail(c, LGT_EINVAL, "lgt_cg_mixed: null pointer");
    if (!(tol >= 0.0) || max_iter < 0 || !(inner_tol > 0.0 && inner_tol < 1.0)) return fail(c, LGT_EINVAL, "lgt_cg_mixed: bad tol / max_iter / inner_tol");
    if (c->prec != LGT_F64) return fail(c, LGT_EINVAL, "lgt_cg_mixed: needs an LGT_F64 handle");
    int rc;
    if ((rc = DISPATCH(c, to_native, c, b, c->ws[5], 12)) != LGT_OK) return rc;
    const double keep = c->inner_tol;
    c->inner_tol = inner_tol;
    int conv = cg_mixed(c, c->ws[5], c->ws[0], nullptr, tol, max_iter, inner_iters, rel_resid);
    c->inner_tol = keep;
    if (outer_cycles) *outer_cycles = c->last_outer;
    if (conv != LGT_OK && conv != LGT_ENOCONV) return conv;
    if ((rc = DISPATCH(c, from_native, c, c->ws[0], x, 12)) != LGT_OK) return rc;
    return conv;
}

// ---- forces
int lgt_gauge_force(lgt_ctx* c, void* F) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!F) return fail(c, LGT_EINVAL, "lgt_gauge_force: null pointer");
    int rc;
    if ((rc = ensure_force_buf(c)) != LGT_OK) return rc;
    if ((rc = DISPATCH(c, gauge_force, c, c->F, 0, 0.0)) != LGT_OK) return rc;
    return DISPATCH(c, momenta_from_native, c, c->F, F);
}
int lgt_gauge_force_accumulate(lgt_ctx* c, double eps) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    return DISPATCH(c, gauge_force, c, c->P, 1, eps);
}
int lgt_fermion_force(lgt_ctx* c, const void* X, const void* Y, void* F, double tol, int max_iter, int* cg_iters) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!F) return fail(c, LGT_EINVAL, "lgt_fermion_force: null pointer");
    if ((X == nullptr) != (Y == nullptr)) return fail(c, LGT_EINVAL, "lgt_fermion_force: give both X and Y or neither");
    int rc, conv = LGT_OK, it = 0;
    if ((rc = ensure_force_buf(c)) != LGT_OK) return rc;
    if (X) {
        if ((rc = DISPATCH(c, to_native, c, X, c->ws[0], 12)) != LGT_OK) return rc;
        if ((rc = DISPATCH(c, to_native, c, Y, c->ws[3], 12)) != LGT_OK) return rc;
    } else {
        if (!c->has_phi) return fail(c, LGT_ESTATE, "lgt_fermion_force: no pseudofermion set");
        conv = solve(c, true, tol, max_iter, &it, nullptr);
        if (conv != LGT_OK && conv != LGT_ENOCONV) return conv;
    }
    if (cg_iters) *cg_iters = it;
    if ((rc = DISPATCH(c, fermion_force, c, c->ws[0], c->ws[3], c->F, 0, 0.0)) != LGT_OK) return rc;
    if ((rc = DISPATCH(c, momenta_from_native, c, c->F, F)) != LGT_OK) return rc;
    return conv;
}
int lgt_fermion_force_native(lgt_ctx* c, const void* X, const void* Y, double eps) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!X || !Y) return fail(c, LGT_EINVAL, "lgt_fermion_force_native: null pointer");
    p_ready(c);
    return DISPATCH(c, fermion_force, c, X, Y, c->P, 1, eps);
}

// ---- molecular dynamics
int lgt_md_kick(lgt_ctx* c, double eps, double tol, int max_iter, int* cg_iters) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    return kick(c, eps, tol, max_iter, cg_iters);
}
int lgt_md_drift(lgt_ctx* c, double eps) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    return DISPATCH(c, link_update, c, eps);
}
int lgt_md_step(lgt_ctx* c, double dt, double tol, int max_iter, int* cg_iters) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    int rc, it1 = 0, it2 = 0, conv = LGT_OK;
    rc = kick(c, 0.5 * dt, tol, max_iter, &it1);
    if (rc == LGT_ENOCONV) conv = rc; else if (rc != LGT_OK) return rc;
    if ((rc = DISPATCH(c, link_update, c, dt)) != LGT_OK) return rc;
    rc = kick(c, 0.5 * dt, tol, max_iter, &it2);
    if (rc == LGT_ENOCONV) conv = rc; else if (rc != LGT_OK) return rc;
    if (cg_iters) *cg_iters = it1 + it2;
    return conv;
}
int lgt_md_trajectory(lgt_ctx* c, int nsteps, double dt, double tol, int max_iter, double* H_initial, double* H_final,
                      long* cg_iters) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (nsteps < 0) return fail(c, LGT_EINVAL, "lgt_md_trajectory: nsteps < 0");
    int rc, it = 0, conv = LGT_OK;
    long total = 0;
    double sg, sf, k;
    if (H_initial) {
        rc = hamiltonian(c, tol, max_iter, &sg, &sf, &k, &it);
        if (rc == LGT_ENOCONV) conv = rc; else if (rc != LGT_OK) return rc;
        *H_initial = k + sg + sf;
    }
    rc = integrate(c, nsteps, dt, tol, max_iter, &total);
    if (rc == LGT_ENOCONV) conv = rc; else if (rc != LGT_OK) return rc;
    if (H_final) {
        rc = hamiltonian(c, tol, max_iter, &sg, &sf, &k, &it);
        if (rc == LGT_ENOCONV) conv = rc; else if (rc != LGT_OK) return rc;
        *H_final = k + sg + sf;
    }
    if (cg_iters) *cg_iters = total;
    CU(cudaStreamSynchronize(c->stream));
    return conv;
}

// ---- HMC around the MD trajectory
int lgt_set_integrator(lgt_ctx* c, int integrator, int n_inner) {
    CHECK_CTX(c);
    if (integrator != LGT_INT_LEAPFROG && integrator != LGT_INT_OMELYAN && integrator != LGT_INT_SEXTON_WEINGARTEN)
        return fail(c, LGT_EINVAL, "lgt_set_integrator: unknown integrator");
    if (integrator == LGT_INT_SEXTON_WEINGARTEN && n_inner < 1) return fail(c, LGT_EINVAL, "lgt_set_integrator: n_inner must be >= 1");
    c->integrator = integrator;
    c->n_inner = integrator == LGT_INT_SEXTON_WEINGARTEN ? n_inner : 1;
    return LGT_OK;
}
int lgt_momentum_heatbath(lgt_ctx* c, unsigned long long seed, unsigned trajectory) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    return DISPATCH(c, momentum_heatbath, c, seed, trajectory);
}
int lgt_pseudofermion_heatbath(lgt_ctx* c, unsigned long long seed, unsigned trajectory, double* eta_norm2) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (c->kappa == 0.0) return fail(c, LGT_ESTATE, "lgt_pseudofermion_heatbath: kappa == 0, no fermions on this handle");
    int rc = DISPATCH(c, pseudofermion_heatbath, c, seed, trajectory, c->scal + 4);
    if (rc != LGT_OK) return rc;
    if (eta_norm2) {
        if ((rc = read_scalars(c, 5)) != LGT_OK) return rc;
        *eta_norm2 = c->h_scal[4];
    }
    return LGT_OK;
}
int lgt_get_pseudofermion(lgt_ctx* c, void* phi) {
    CHECK_CTX(c);
    if (!phi) return fail(c, LGT_EINVAL, "lgt_get_pseudofermion: null pointer");
    if (!c->has_phi) return fail(c, LGT_ESTATE, "lgt_get_pseudofermion: no pseudofermion set");
    return DISPATCH(c, from_native, c, c->phi, phi, 12);
}
int lgt_hmc_trajectory(lgt_ctx* c, int nsteps, double dt, double tol, int max_iter, unsigned long long seed, unsigned trajectory,
                       double* dH, int* accepted, long* cg_iters, double* H_initial) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (nsteps < 0) return fail(c, LGT_EINVAL, "lgt_hmc_trajectory: nsteps < 0");
    int rc, it = 0, conv = LGT_OK;
    long total = 0;
    const bool ferm = c->kappa != 0.0;
    if (!c->Usave) CU(cudaMalloc(&c->Usave, links_bytes(c)));
    if ((rc = DISPATCH(c, momentum_heatbath, c, seed, trajectory)) != LGT_OK) return rc;
    if (ferm && (rc = DISPATCH(c, pseudofermion_heatbath, c, seed, trajectory, c->scal + 4)) != LGT_OK) return rc;
    CU(cudaMemcpyAsync(c->Usave, c->U, links_bytes(c), cudaMemcpyDeviceToDevice, c->stream));
    if ((rc = DISPATCH(c, plaquette_sum, c, c->scal + 0)) != LGT_OK) return rc;
    if ((rc = DISPATCH(c, kinetic, c, c->scal + 1)) != LGT_OK) return rc;
    if ((rc = read_scalars(c, 5)) != LGT_OK) return rc;
    // S_F at the start is |eta|^2 exactly (phi = D^dag eta), no solve needed
    const double H0 = c->h_scal[1] + c->beta * (6.0 * (double)c->g.V - c->h_scal[0]) + (ferm ? c->h_scal[4] : 0.0);
    rc = integrate(c, nsteps, dt, tol, max_iter, &total);
    if (rc == LGT_ENOCONV) conv = rc; else if (rc != LGT_OK) return rc;
    double sg, sf, k;
    rc = hamiltonian(c, tol, max_iter, &sg, &sf, &k, &it);
    if (rc == LGT_ENOCONV) conv = rc; else if (rc != LGT_OK) return rc;
    total += it;
    const double d = (k + sg + sf) - H0;
    const bool acc = metropolis_uniform(seed, trajectory) < exp(-d);
    if (!acc) {
        CU(cudaMemcpyAsync(c->U, c->Usave, links_bytes(c), cudaMemcpyDeviceToDevice, c->stream));
        c->u32_valid = false;
    c->usm_valid = false;
    if (c->dd_links_valid) *c->dd_links_valid = false;
        c->ucb_valid = false;
    c->ucb32_valid = false;
    c->inner_exact = false;
    }
    CU(cudaStreamSynchronize(c->stream));
    if (dH) *dH = d;
    if (accepted) *accepted = acc ? 1 : 0;
    if (cg_iters) *cg_iters = total;
    if (H_initial) *H_initial = H0;
    return conv;
}

// ---- measured roofline denominators ("the builder must microbenchmark" the fp64 FMA peak)
int lgt_measure_peaks(lgt_ctx* c, int launches, double* fma_tflops_best, double* fma_tflops_mean, double* copy_gbs_best,
                      double* copy_gbs_mean) {
    CHECK_CTX(c);
    if (launches < 1 || launches > 1000) return fail(c, LGT_EINVAL, "lgt_measure_peaks: launches must be in 1..1000");
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    int rc = LGT_OK;
    auto time_launches = [&](auto launch, double work_per_launch, double* best, double* mean) -> int {
        double tb = 1e30, tsum = 0.0;
        for (int i = -2; i < launches; i++) {  // two untimed launches first
            CU(cudaEventRecord(e0, c->stream));
            launch();
            CU(cudaEventRecord(e1, c->stream));
            CU(cudaEventSynchronize(e1));
            CU(cudaGetLastError());
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, e0, e1));
            if (i < 0) continue;
            tsum += ms;
            if (ms < tb) tb = ms;
        }
        if (best) *best = work_per_launch / (tb * 1e-3);
        if (mean) *mean = work_per_launch / (tsum / launches * 1e-3);
        return LGT_OK;
    };
    if (fma_tflops_best || fma_tflops_mean) {
        // every SM holds 8 blocks of 256 threads (64 warps: full occupancy), each thread PEAK_CHAINS independent chains
        const int grid = sms * 8, iters = c->prec == LGT_F64 ? 4096 : 16384;
        const double flops = 2.0 * PEAK_CHAINS * (double)iters * 256.0 * grid;
        double* sink = c->partials;  // grid <= red_blocks + 64 doubles... one slot per block
        if (c->prec == LGT_F64)
            rc = time_launches([&]() { peak_fma_kernel<double><<<grid, 256, 0, c->stream>>>(sink, iters, 1.0000001, 1e-9); }, flops * 1e-12,
                               fma_tflops_best, fma_tflops_mean);
        else
            rc = time_launches([&]() { peak_fma_kernel<float><<<grid, 256, 0, c->stream>>>(sink, iters, 1.0001f, 1e-6f); }, flops * 1e-12,
                               fma_tflops_best, fma_tflops_mean);
        c->launches += launches + 2;
    }
    if (rc == LGT_OK && (copy_gbs_best || copy_gbs_mean)) {
        // a plain copy of the native link field (604 MB at 32^4 fp64, well beyond L2) into a scratch buffer
        const size_t bytes = links_bytes(c);
        void* dst = nullptr;
        cudaError_t e = cudaMalloc(&dst, bytes);
        if (e != cudaSuccess) rc = fail(c, LGT_ENOMEM, "lgt_measure_peaks: cudaMalloc", e);
        else {
            const size_t n16 = bytes / 16;
            rc = time_launches([&]() { peak_copy_kernel<<<sms * 16, 256, 0, c->stream>>>((const int4*)c->U, (int4*)dst, n16); }, 2.0 * (double)bytes * 1e-9,
                               copy_gbs_best, copy_gbs_mean);
            c->launches += launches + 2;
            cudaFree(dst);
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}

// ---- stout smearing
int lgt_set_smearing(lgt_ctx* c, int n_levels, double rho) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (n_levels < 0 || n_levels > LGT_MAX_SMEAR) return fail(c, LGT_EINVAL, "lgt_set_smearing: n_levels must be in 0..8");
    if (n_levels > 0 && !(rho >= 0.0)) return fail(c, LGT_EINVAL, "lgt_set_smearing: rho must be >= 0");
    c->nsmear = n_levels;
    c->rho = n_levels ? rho : 0.0;
    c->usm_valid = false;
    if (c->dd_links_valid) *c->dd_links_valid = false;
    c->u32_valid = false;
    c->ucb_valid = false;
    c->ucb32_valid = false;
    c->inner_exact = false;
    return LGT_OK;
}
int lgt_get_smeared_links(lgt_ctx* c, void* U) {
    CHECK_CTX(c);
    NOT_SLAB(c);
    if (!U) return fail(c, LGT_EINVAL, "lgt_get_smeared_links: null pointer");
    int rc = DISPATCH(c, ensure_fermion_links, c);
    if (rc != LGT_OK) return rc;
    return DISPATCH(c, from_native, c, c->Uf, U, 36);
}

}  // extern "C"

#include "lgt_dd.cuh"
