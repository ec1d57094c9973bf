// lgt_dd.cuh -- the MD step on a lattice decomposed into time slabs, one slab per rank (include/lgt.h "lgt_dd_*",
// SURVEY.md 8(e)).  Included by lgt_api.cu; uses its handle, launch macro and Ops<T>.
//
// A rank's slab is an ordinary handle on the local lattice (Lx, Ly, Lz, Lt_local + 2): slices 0 and Lt_local + 1
// are ghost copies of the neighbour ranks' boundary slices, and Geom::s_begin / s_end restrict every compute kernel
// to the interior.  Because t is the slowest index and Lx Ly Lz is a multiple of 32, a time slice of any native field
// is one contiguous run, so a halo exchange is two sends and two receives per rank and field, with no packing kernel.
// The same driver serves three transports: NCCL send/recv + all-reduce between processes (one rank per process); a
// caller-supplied HOST transport (two callbacks: a paired send/receive of host buffers and an all-reduce of host
// doubles -- MPI, gloo, ...; slices are staged through pinned memory), also one rank per process; and plain device
// copies between ranks that live in this process (all ranks of the group on one device and one stream, stepped in
// lockstep, nothing ever waits on another rank).  All three issue the sends and receives of lgt_dd_halo_plan in the
// same order.
#pragma once
#include <dlfcn.h>

namespace {

// ---- NCCL through dlopen: no link-time dependency, and the process's already loaded libnccl.so.2 (torch's) is reused
struct NcclApi {
    typedef struct { char internal[128]; } UniqueId;
    void* lib = nullptr;
    int (*GetUniqueId)(UniqueId*) = nullptr;
    int (*CommInitRank)(void**, int, UniqueId, int) = nullptr;
    int (*CommDestroy)(void*) = nullptr;
    int (*GroupStart)() = nullptr;
    int (*GroupEnd)() = nullptr;
    int (*Send)(const void*, size_t, int, int, void*, cudaStream_t) = nullptr;
    int (*Recv)(void*, size_t, int, int, void*, cudaStream_t) = nullptr;
    int (*AllReduce)(const void*, void*, size_t, int, int, void*, cudaStream_t) = nullptr;
    const char* (*GetErrorString)(int) = nullptr;
    bool load() {
        if (lib) return true;
        lib = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
        if (!lib) lib = dlopen("libnccl.so", RTLD_NOW | RTLD_GLOBAL);
        if (!lib) return false;
#define NCCL_SYM(name) *(void**)(&name) = dlsym(lib, "nccl" #name)
        NCCL_SYM(GetUniqueId);
        NCCL_SYM(CommInitRank);
        NCCL_SYM(CommDestroy);
        NCCL_SYM(GroupStart);
        NCCL_SYM(GroupEnd);
        NCCL_SYM(Send);
        NCCL_SYM(Recv);
        NCCL_SYM(AllReduce);
        NCCL_SYM(GetErrorString);
#undef NCCL_SYM
        return GetUniqueId && CommInitRank && CommDestroy && GroupStart && GroupEnd && Send && Recv && AllReduce;
    }
};
NcclApi g_nccl;
constexpr int NCCL_CHAR = 0, NCCL_DOUBLE = 8, NCCL_SUM = 0;  // ncclDataType_t / ncclRedOp_t values of nccl.h

std::string g_dd_create_error;

}  // namespace

struct lgt_dd {
    int nranks = 0;
    std::vector<lgt_ctx*> rk;   // this process's ranks
    std::vector<int> rank_of;   // their global rank numbers
    int Lt_loc = 0;
    int V3 = 0;
    int prec = LGT_F64;
    int device = 0;
    cudaStream_t stream = nullptr;
    bool links_ghost_valid = false;
    // (Pt, Pz) grid (lgt_dd_create_grid): Pz > 0; rank = pt * Pz + pz; every rank then also has two ghost z planes and
    // V3 counts them (it is the size of a LOCAL time slice).  Time slabs: Pz = 0.
    int Pt = 0, Pz = 0, Lz_loc = 0, LxLy = 0;
    long long Vglob = 0;
    void* d_stage = nullptr;  // device staging of the z faces for NCCL (2 outgoing, 2 incoming)
    size_t d_stage_bytes = 0;
    void* comm = nullptr;  // ncclComm_t; null: host transport, or every rank is local
    // host transport (lgt_dd_set_host_transport): callbacks + pinned staging (2 outgoing, 2 incoming slices; sums)
    lgt_dd_sendrecv_fn host_sendrecv = nullptr;
    lgt_dd_allreduce_fn host_allreduce = nullptr;
    void* host_user = nullptr;
    char* h_stage = nullptr;
    size_t h_stage_bytes = 0;
    double* h_sum = nullptr;
    // LGT_DD_PUSH: halos of the CG fields t (ws[3]) and r (ws[1]) are stored into the neighbours' ghost slices by the
    // producing kernels.  Neighbours in other processes: their buffers mapped through CUDA IPC, [field r, t][lo, hi].
    int halo_mode = 0;
    // LGT_DD_OVERLAP: the exchange runs on its own stream while the slab's bulk is computed (lazy)
    cudaStream_t halo_stream = nullptr;
    cudaEvent_t ev_ready = nullptr, ev_halo = nullptr;
    // LGT_DD_HALF: per local rank one buffer of four half-spinor faces [lo_out | hi_out | hi_in | lo_in], 6 V3 complex each (lazy)
    std::vector<void*> half_faces;
    size_t half_face_bytes = 0;
    void* ipc_peer[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};
    bool ipc_open[2][2] = {{false, false}, {false, false}};
    std::string err;
};

namespace {

int dd_fail(lgt_dd* d, int code, const char* what, const char* detail = nullptr) {
    std::string m = what;
    if (detail && *detail) m += std::string(": ") + detail;
    if (d) d->err = m;
    else g_dd_create_error = m;
    return code;
}
#define DD_CU(call)                                                                        \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess) return dd_fail(d, LGT_ECUDA, #call, cudaGetErrorString(e_)); \
    } while (0)
#define DD_NCCL(call)                                                                                              \
    do {                                                                                                           \
        int r_ = (call);                                                                                           \
        if (r_ != 0) return dd_fail(d, LGT_ECUDA, #call, g_nccl.GetErrorString ? g_nccl.GetErrorString(r_) : ""); \
    } while (0)
// a failing rank-level call: carry its message up
#define DD_RK(i, call)                                                     \
    do {                                                                   \
        int rc_ = (call);                                                  \
        if (rc_ != LGT_OK) return dd_fail(d, rc_, d->rk[i]->err.c_str()); \
    } while (0)

int dd_local_index(const lgt_dd* d, int rank) {
    for (size_t i = 0; i < d->rank_of.size(); i++)
        if (d->rank_of[i] == rank) return (int)i;
    return -1;
}

// The halo plan of one rank (include/lgt.h "lgt_dd_halo_plan"): rank r's first interior slice (local slice 1) goes to
// the upper ghost slice (Lt_loc + 1) of rank r - 1, its last interior slice (Lt_loc) to the lower ghost slice (0) of
// rank r + 1, periodic in ranks.  Every transport issues the two sends and the two receives in THIS order; sends and
// receives between one pair of ranks are matched in issue order (NCCL, MPI and gloo all guarantee that), which is what
// makes nranks = 2 (both neighbours are the one other rank) and nranks = 1 (a rank is its own neighbour) come out right.
struct HaloPlan {
    int send_peer[2], send_slice[2], recv_peer[2], recv_slice[2];
};
HaloPlan halo_plan(int nranks, int rank, int lt_loc) {
    HaloPlan p;
    const int dn = (rank + nranks - 1) % nranks, up = (rank + 1) % nranks;
    p.send_peer[0] = dn;
    p.send_slice[0] = 1;
    p.send_peer[1] = up;
    p.send_slice[1] = lt_loc;
    p.recv_peer[0] = up;
    p.recv_slice[0] = lt_loc + 1;
    p.recv_peer[1] = dn;
    p.recv_slice[1] = 0;
    return p;
}

// A group that owns fewer ranks than the lattice has needs a transport before anything can be exchanged or summed.
int dd_need_transport(lgt_dd* d) {
    if (d->rk.size() != (size_t)d->nranks && !d->comm && !d->host_sendrecv)
        return dd_fail(d, LGT_ESTATE, "this group holds one of several ranks and has no transport yet: call lgt_dd_nccl_init or "
                                      "lgt_dd_set_host_transport first");
    return LGT_OK;
}

int dd_host_stage(lgt_dd* d, size_t bytes) {
    if (d->h_stage_bytes >= bytes) return LGT_OK;
    DD_CU(cudaStreamSynchronize(d->stream));
    if (d->h_stage) cudaFreeHost(d->h_stage);
    d->h_stage = nullptr;
    d->h_stage_bytes = 0;
    DD_CU(cudaMallocHost((void**)&d->h_stage, bytes));
    d->h_stage_bytes = bytes;
    return LGT_OK;
}

// ---- (Pt, Pz) grid: the halo of one split direction as two strided regions out, two in ("first T, then Z").
// t: whole local time slices (one contiguous run each, z ghost planes included).  z: the xy planes z = 1 and z = Lz_loc of
// EVERY local time slice, ghost slices included -- an xy plane is Lx*Ly/32 whole layout blocks, so a z face is Lt_loc + 2
// contiguous runs at the pitch of a time slice and moves by 2-D copies, again without a packing kernel.  Doing t first
// and z second fills the corners: the z neighbour's ghost time slices already hold the diagonal rank's planes, which is what
// the staples U_nu(x + mu - nu) need.
struct GridHalo {
    int dn, up;            // peers: my first interior region goes to dn's upper ghost, my last to up's lower ghost
    size_t send_off[2], recv_off[2];  // bytes from the field's base: sends (to dn, to up), receives (from up, from dn)
    size_t width, pitch;   // bytes per run, distance between runs
    int height;            // runs
};
GridHalo grid_halo(const lgt_dd* d, int rank, int dim /* 0: t, 1: z */, int per_site, size_t esize) {
    GridHalo h;
    const int pt = rank / d->Pz, pz = rank % d->Pz;
    const size_t slice = (size_t)d->V3 * per_site * esize;
    if (dim == 0) {
        h.dn = ((pt + d->Pt - 1) % d->Pt) * d->Pz + pz;
        h.up = ((pt + 1) % d->Pt) * d->Pz + pz;
        h.width = slice;
        h.pitch = slice;
        h.height = 1;
        h.send_off[0] = slice;
        h.send_off[1] = (size_t)d->Lt_loc * slice;
        h.recv_off[0] = (size_t)(d->Lt_loc + 1) * slice;
        h.recv_off[1] = 0;
    } else {
        h.dn = pt * d->Pz + (pz + d->Pz - 1) % d->Pz;
        h.up = pt * d->Pz + (pz + 1) % d->Pz;
        h.width = (size_t)d->LxLy * per_site * esize;
        h.pitch = slice;
        h.height = d->Lt_loc + 2;
        h.send_off[0] = h.width;
        h.send_off[1] = (size_t)d->Lz_loc * h.width;
        h.recv_off[0] = (size_t)(d->Lz_loc + 1) * h.width;
        h.recv_off[1] = 0;
    }
    return h;
}
int dd_host_stage(lgt_dd* d, size_t bytes);
int dd_exchange_grid(lgt_dd* d, void* const* base, int per_site, size_t esize) {
    const int n = (int)d->rk.size();
    for (int dim = 0; dim < 2; dim++) {
        if (!d->comm && !d->host_sendrecv) {  // every rank in this process: device copies
            for (int i = 0; i < n; i++) {
                const GridHalo h = grid_halo(d, d->rank_of[i], dim, per_site, esize);
                const int peers[2] = {h.dn, h.up};
                for (int k = 0; k < 2; k++) {
                    const int peer = dd_local_index(d, peers[k]);
                    if (peer < 0) return dd_fail(d, LGT_ESTATE, "dd_exchange: a neighbour rank is not in this process");
                    // my k-th send lands where the peer receives its k-th message (send 0, to dn, is dn's receive 0, from its up)
                    DD_CU(cudaMemcpy2DAsync((char*)base[peer] + h.recv_off[k], h.pitch, (const char*)base[i] + h.send_off[k], h.pitch, h.width,
                                            h.height, cudaMemcpyDeviceToDevice, d->stream));
                }
            }
            continue;
        }
        const GridHalo h = grid_halo(d, d->rank_of[0], dim, per_site, esize);
        const size_t bytes = h.width * h.height;
        const int send_peer[2] = {h.dn, h.up}, recv_peer[2] = {h.up, h.dn};
        char* mine = (char*)base[0];
        if (d->comm) {
            if (d->d_stage_bytes < 4 * bytes) {
                DD_CU(cudaStreamSynchronize(d->stream));
                if (d->d_stage) cudaFree(d->d_stage);
    if (d->halo_stream) cudaStreamDestroy(d->halo_stream);
    for (void* f : d->half_faces) cudaFree(f);
    if (d->ev_ready) cudaEventDestroy(d->ev_ready);
    if (d->ev_halo) cudaEventDestroy(d->ev_halo);
                d->d_stage = nullptr;
                d->d_stage_bytes = 0;
                DD_CU(cudaMalloc(&d->d_stage, 4 * bytes));
                d->d_stage_bytes = 4 * bytes;
            }
            char* st = (char*)d->d_stage;
            for (int k = 0; k < 2; k++)
                DD_CU(cudaMemcpy2DAsync(st + k * bytes, h.width, mine + h.send_off[k], h.pitch, h.width, h.height, cudaMemcpyDeviceToDevice, d->stream));
            DD_NCCL(g_nccl.GroupStart());
            for (int k = 0; k < 2; k++) DD_NCCL(g_nccl.Send(st + k * bytes, bytes, NCCL_CHAR, send_peer[k], d->comm, d->stream));
            for (int k = 0; k < 2; k++) DD_NCCL(g_nccl.Recv(st + (2 + k) * bytes, bytes, NCCL_CHAR, recv_peer[k], d->comm, d->stream));
            DD_NCCL(g_nccl.GroupEnd());
            for (int k = 0; k < 2; k++)
                DD_CU(cudaMemcpy2DAsync(mine + h.recv_off[k], h.pitch, st + (2 + k) * bytes, h.width, h.width, h.height, cudaMemcpyDeviceToDevice, d->stream));
            continue;
        }
        int rc;
        if ((rc = dd_host_stage(d, 4 * bytes)) != LGT_OK) return rc;
        char* hs = d->h_stage;
        for (int k = 0; k < 2; k++)
            DD_CU(cudaMemcpy2DAsync(hs + k * bytes, h.width, mine + h.send_off[k], h.pitch, h.width, h.height, cudaMemcpyDeviceToHost, d->stream));
        DD_CU(cudaStreamSynchronize(d->stream));
        const void* const sb[2] = {hs, hs + bytes};
        void* const rb[2] = {hs + 2 * bytes, hs + 3 * bytes};
        if (d->host_sendrecv(d->host_user, sb, send_peer, rb, recv_peer, bytes) != 0)
            return dd_fail(d, LGT_ECUDA, "dd_exchange: the host transport's send/receive callback failed");
        for (int k = 0; k < 2; k++)
            DD_CU(cudaMemcpy2DAsync(mine + h.recv_off[k], h.pitch, hs + (2 + k) * bytes, h.width, h.width, h.height, cudaMemcpyHostToDevice, d->stream));
        DD_CU(cudaStreamSynchronize(d->stream));  // the staging buffer is reused by the z phase
    }
    return LGT_OK;
}

// Halo exchange of one native field per local rank: base[i] points to the field of local rank i, `per_site` = complex
// (or pair) elements per site (12 spinor, 36 links, 16 compact momenta).
int dd_exchange(lgt_dd* d, void* const* base, int per_site, size_t esize = 0) {
    if (!esize) esize = d->prec == LGT_F64 ? 16 : 8;
    if (d->Pz > 0) {
        int rcg = dd_need_transport(d);
        return rcg != LGT_OK ? rcg : dd_exchange_grid(d, base, per_site, esize);
    }
    const size_t slice = (size_t)d->V3 * per_site * esize;
    const int n = (int)d->rk.size();
    int rc;
    if ((rc = dd_need_transport(d)) != LGT_OK) return rc;
    if (!d->comm && !d->host_sendrecv) {
        for (int i = 0; i < n; i++) {
            const HaloPlan p = halo_plan(d->nranks, d->rank_of[i], d->Lt_loc);
            char* mine = (char*)base[i];
            for (int k = 0; k < 2; k++) {
                // my k-th send lands where the peer's plan receives from me in the same position: send 0 (to r - 1) is
                // that rank's receive 0 (from its r + 1), send 1 (to r + 1) its receive 1
                const int peer = dd_local_index(d, p.send_peer[k]);
                if (peer < 0) return dd_fail(d, LGT_ESTATE, "dd_exchange: a neighbour rank is not in this process");
                const HaloPlan q = halo_plan(d->nranks, p.send_peer[k], d->Lt_loc);
                DD_CU(cudaMemcpyAsync((char*)base[peer] + (size_t)q.recv_slice[k] * slice, mine + (size_t)p.send_slice[k] * slice, slice,
                                      cudaMemcpyDeviceToDevice, d->stream));
            }
        }
        return LGT_OK;
    }
    // one rank per process
    const HaloPlan p = halo_plan(d->nranks, d->rank_of[0], d->Lt_loc);
    char* mine = (char*)base[0];
    if (d->comm) {
        DD_NCCL(g_nccl.GroupStart());
        for (int k = 0; k < 2; k++) DD_NCCL(g_nccl.Send(mine + (size_t)p.send_slice[k] * slice, slice, NCCL_CHAR, p.send_peer[k], d->comm, d->stream));
        for (int k = 0; k < 2; k++) DD_NCCL(g_nccl.Recv(mine + (size_t)p.recv_slice[k] * slice, slice, NCCL_CHAR, p.recv_peer[k], d->comm, d->stream));
        DD_NCCL(g_nccl.GroupEnd());
        return LGT_OK;
    }
    // host transport: outgoing slices to pinned memory, the caller's paired send/receive, incoming slices back
    if ((rc = dd_host_stage(d, 4 * slice)) != LGT_OK) return rc;
    char* h = d->h_stage;
    for (int k = 0; k < 2; k++)
        DD_CU(cudaMemcpyAsync(h + k * slice, mine + (size_t)p.send_slice[k] * slice, slice, cudaMemcpyDeviceToHost, d->stream));
    DD_CU(cudaStreamSynchronize(d->stream));  // also orders the previous exchange's upload before the buffers are reused
    const void* const sb[2] = {h, h + slice};
    void* const rb[2] = {h + 2 * slice, h + 3 * slice};
    if (d->host_sendrecv(d->host_user, sb, p.send_peer, rb, p.recv_peer, slice) != 0)
        return dd_fail(d, LGT_ECUDA, "dd_exchange: the host transport's send/receive callback failed");
    for (int k = 0; k < 2; k++)
        DD_CU(cudaMemcpyAsync(mine + (size_t)p.recv_slice[k] * slice, h + (2 + k) * slice, slice, cudaMemcpyHostToDevice, d->stream));
    return LGT_OK;
}

// The same plan for two arbitrary regions per rank (time slabs): rank r's region send_off[0] goes to rank r - 1 and lands at
// its recv_off[0], send_off[1] goes to rank r + 1 and lands at its recv_off[1]; `bytes` each.  Used for the half-spinor faces.
int dd_exchange_regions(lgt_dd* d, void* const* base, const size_t send_off[2], const size_t recv_off[2], size_t bytes) {
    const int n = (int)d->rk.size();
    int rc;
    if ((rc = dd_need_transport(d)) != LGT_OK) return rc;
    if (!d->comm && !d->host_sendrecv) {
        for (int i = 0; i < n; i++) {
            const HaloPlan p = halo_plan(d->nranks, d->rank_of[i], d->Lt_loc);
            for (int k = 0; k < 2; k++) {
                const int peer = dd_local_index(d, p.send_peer[k]);
                if (peer < 0) return dd_fail(d, LGT_ESTATE, "dd_exchange: a neighbour rank is not in this process");
                DD_CU(cudaMemcpyAsync((char*)base[peer] + recv_off[k], (const char*)base[i] + send_off[k], bytes, cudaMemcpyDeviceToDevice, d->stream));
            }
        }
        return LGT_OK;
    }
    const HaloPlan p = halo_plan(d->nranks, d->rank_of[0], d->Lt_loc);
    char* mine = (char*)base[0];
    if (d->comm) {
        DD_NCCL(g_nccl.GroupStart());
        for (int k = 0; k < 2; k++) DD_NCCL(g_nccl.Send(mine + send_off[k], bytes, NCCL_CHAR, p.send_peer[k], d->comm, d->stream));
        for (int k = 0; k < 2; k++) DD_NCCL(g_nccl.Recv(mine + recv_off[k], bytes, NCCL_CHAR, p.recv_peer[k], d->comm, d->stream));
        DD_NCCL(g_nccl.GroupEnd());
        return LGT_OK;
    }
    if ((rc = dd_host_stage(d, 4 * bytes)) != LGT_OK) return rc;
    char* h = d->h_stage;
    for (int k = 0; k < 2; k++) DD_CU(cudaMemcpyAsync(h + k * bytes, mine + send_off[k], bytes, cudaMemcpyDeviceToHost, d->stream));
    DD_CU(cudaStreamSynchronize(d->stream));
    const void* const sb[2] = {h, h + bytes};
    void* const rb[2] = {h + 2 * bytes, h + 3 * bytes};
    if (d->host_sendrecv(d->host_user, sb, p.send_peer, rb, p.recv_peer, bytes) != 0)
        return dd_fail(d, LGT_ECUDA, "dd_exchange: the host transport's send/receive callback failed");
    for (int k = 0; k < 2; k++) DD_CU(cudaMemcpyAsync(mine + recv_off[k], h + (2 + k) * bytes, bytes, cudaMemcpyHostToDevice, d->stream));
    DD_CU(cudaStreamSynchronize(d->stream));  // the staging buffer is reused by the next exchange
    return LGT_OK;
}

// Sum of `count` doubles over all ranks, in place at ptr[i] of every local rank (device memory).
int dd_allreduce(lgt_dd* d, double* const* ptr, int count) {
    int rc;
    if ((rc = dd_need_transport(d)) != LGT_OK) return rc;
    if (d->comm) {
        DD_NCCL(g_nccl.AllReduce(ptr[0], ptr[0], (size_t)count, NCCL_DOUBLE, NCCL_SUM, d->comm, d->stream));
        return LGT_OK;
    }
    if (d->host_allreduce) {
        if (count > 8) return dd_fail(d, LGT_EINVAL, "dd_allreduce: at most 8 doubles");
        if (!d->h_sum) DD_CU(cudaMallocHost((void**)&d->h_sum, 8 * sizeof(double)));
        DD_CU(cudaMemcpyAsync(d->h_sum, ptr[0], count * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
        DD_CU(cudaStreamSynchronize(d->stream));
        if (d->host_allreduce(d->host_user, d->h_sum, count) != 0)
            return dd_fail(d, LGT_ECUDA, "dd_allreduce: the host transport's all-reduce callback failed");
        DD_CU(cudaMemcpyAsync(ptr[0], d->h_sum, count * sizeof(double), cudaMemcpyHostToDevice, d->stream));
        DD_CU(cudaStreamSynchronize(d->stream));  // h_sum is reused by the next sum
        return LGT_OK;
    }
    DdPtrs p;
    for (size_t i = 0; i < 8; i++) p.p[i] = i < d->rk.size() ? ptr[i] : nullptr;
    dd_local_allreduce_kernel<<<1, 32, 0, d->stream>>>(p, (int)d->rk.size(), count);
    DD_CU(cudaGetLastError());
    return LGT_OK;
}

int dd_exchange_links(lgt_dd* d) {
    if (d->links_ghost_valid) return LGT_OK;
    std::vector<void*> u;
    for (lgt_ctx* c : d->rk) u.push_back(c->U);
    int rc = dd_exchange(d, u.data(), 36);
    if (rc == LGT_OK) d->links_ghost_valid = true;
    return rc;
}

}  // namespace

namespace {

// (D^dag D) x = b with the group's solver (plain CG, or the mixed-precision defect correction on LGT_F64 groups)
int dd_solve(lgt_dd* d, int ib, bool want_y, double tol, int max_iter, int* iters);
// mixed-precision form of the even/odd solve (defined after the driver)
int dd_eo_cg_mixed(lgt_dd* d, double tol, int max_iter, int* iters);

// Where a rank's boundary slices of one field go: the same field of rank r - 1 (its upper ghost slice receives our first
// interior slice) and of rank r + 1 (its lower ghost slice receives our last interior slice).
template <class T> struct Neighbours {
    typename Vec2<T>::type* lo = nullptr;
    typename Vec2<T>::type* hi = nullptr;
};

// The driver: every step loops over the local ranks (one in production, all of them in the single-GPU verification
// mode), then does the step's communication, so that both transports run the same sequence of launches.
template <class T> struct DdOps {
    typedef typename Vec2<T>::type T2;
    typedef Ops<T> O;

    // the ghost z planes of a grid rank stay out of the streaming sums (none on time slabs)
    static ZMask zmask(const lgt_ctx* c) {
        ZMask m;
        if (c->g.z_hi - c->g.z_lo != c->g.L[2]) {
            m.xy = c->g.L[0] * c->g.L[1];
            m.Lz = c->g.L[2];
            m.z_lo = c->g.z_lo;
            m.z_hi = c->g.z_hi;
        }
        return m;
    }
    static size_t spinor_off(const lgt_ctx* c) { return (size_t)12 * c->g.s_begin; }
    static size_t spinor_n(const lgt_ctx* c) { return (size_t)12 * own_sites(c); }

    // Field k of a rank in precision T: 0..5 = ws[k], 6 = phi, 7 = links.  DdOps<float> on an LGT_F64 group is the fp32
    // inner solve of the mixed-precision solver and works on the rank's fp32 copies: links U32 and
    // ws32 = {b, e, r, p, t} standing for the roles ws[5] (b), ws[0] (x), ws[1] (r), ws[2] (p), ws[3] (t).
    static bool fp32_on_f64(const lgt_ctx* c) { return sizeof(T) == 4 && c->prec == LGT_F64; }
    static void* fld(lgt_ctx* c, int k) {
        if (fp32_on_f64(c)) {
            switch (k) {
                case 0: return c->ws32[1];
                case 1: return c->ws32[2];
                case 2: return c->ws32[3];
                case 3: return c->ws32[4];
                case 5: return c->ws32[0];
                case 7: return c->U32;  // fp32 copy of the fermions' links
                default: return nullptr;
            }
        }
        return k == 6 ? c->phi : k == 7 ? c->Uf : c->ws[k];
    }
    static int exchange_spinor(lgt_dd* d, int k) {
        std::vector<void*> f;
        for (lgt_ctx* c : d->rk) f.push_back(fld(c, k));
        return dd_exchange(d, f.data(), 12, sizeof(T2));
    }
    static int allreduce_tmp(lgt_dd* d) {
        std::vector<double*> p;
        for (lgt_ctx* c : d->rk) p.push_back(&c->st->tmp);
        return dd_allreduce(d, p.data(), 1);
    }

    // A pushing stencil launch over the owned range [*begin, *end) of a field with `slice` sites per time slice (a
    // multiple of 128): the two boundary slices first, each with the PUSH kernel and its one target -- the halo stores
    // are then in flight while the bulk computes -- then the interior with the ordinary kernel.  Block partials land
    // where one launch over the whole range would put them, so the sums are unchanged bit for bit.
    // `launch(push)` issues the kernel for the range currently set in c->g / c->partials (push == nullptr: no push).
    template <class Launch>
    static int split_launch(lgt_ctx* c, int* begin, int* end, int slice, int lt_loc, const Neighbours<T>& nb, Launch launch) {
        const int b0 = *begin, e0 = *end;
        double* const part0 = c->partials;
        int rc;
        PushTo<T> to;
        if (lt_loc == 1) {  // the one slice feeds both neighbours
            to.a = nb.lo;
            to.da = slice;
            to.b = nb.hi;
            to.db = -slice;
            return launch(&to);
        }
        *end = b0 + slice;  // first interior slice -> upper ghost slice of rank r - 1
        to.a = nb.lo;
        to.da = lt_loc * slice;
        rc = launch(&to);
        if (rc == LGT_OK) {
            *begin = e0 - slice;  // last interior slice -> lower ghost slice of rank r + 1
            *end = e0;
            c->partials = part0 + (e0 - slice - b0) / 128;
            to.a = nb.hi;
            to.da = -lt_loc * slice;
            rc = launch(&to);
        }
        if (rc == LGT_OK && lt_loc > 2) {
            *begin = b0 + slice;  // the bulk
            *end = e0 - slice;
            c->partials = part0 + slice / 128;
            rc = launch(nullptr);
        }
        *begin = b0;
        *end = e0;
        c->partials = part0;
        return rc;
    }
    static int dslash_pushing(lgt_dd* d, lgt_ctx* c, const void* in, void* out, int dagger, int mode, void* r, const Neighbours<T>& nb) {
        return split_launch(c, &c->g.s_begin, &c->g.s_end, d->V3, d->Lt_loc, nb,
                            [&](const PushTo<T>* push) { return O::dslash(c, fld(c, 7), in, out, dagger, mode, r, push); });
    }

    // LGT_DD_OVERLAP (time slabs, CG loop): the stencil launch over field `k` split so that the halo exchange of `k` runs on
    // the group's halo stream WHILE the bulk of every slab (the slices that touch no ghost slice) is computed; the two
    // boundary slices follow once the halo has landed.  Block partials land where one launch over the slab would put them:
    // the sums, hence the iterates, are bitwise those of LGT_DD_EXCHANGE.  `launch(c)` issues the kernel for the range
    // currently set in c->g / c->partials.
    // LGT_DD_HALF: the same schedule with HALF SPINORS on the wire: halo_pack_kernel projects the first slice
    // and projects and multiplies the last slice of field `k` into two faces of 6 complex per site, the faces travel instead of
    // the 12-complex slices (half the bytes), and the two boundary slices run dslash_halo_kernel, which takes the t hop that
    // reaches into the ghost slice from the received face.  Same operations on the same numbers: bitwise the same iterates.
    // mode 1: t = D p (out = field 3); mode 2: r -= alpha D^dag t (r = field 1).
    // the halo stream with its events, and per local rank four faces of 6 V3 complex doubles (enough for either precision and
    // for the half fields of the even/odd hops)
    static int ensure_half_faces(lgt_dd* d) {
        const int n = (int)d->rk.size();
        const size_t face = (size_t)6 * d->V3 * sizeof(double2);
        if (!d->halo_stream) {
            DD_CU(cudaStreamCreateWithFlags(&d->halo_stream, cudaStreamNonBlocking));
            DD_CU(cudaEventCreateWithFlags(&d->ev_ready, cudaEventDisableTiming));
            DD_CU(cudaEventCreateWithFlags(&d->ev_halo, cudaEventDisableTiming));
        }
        if (d->half_faces.size() != (size_t)n || d->half_face_bytes < face) {
            DD_CU(cudaStreamSynchronize(d->stream));
            for (void* f : d->half_faces) cudaFree(f);
            d->half_faces.assign(n, nullptr);
            for (int i = 0; i < n; i++) DD_CU(cudaMalloc(&d->half_faces[i], 4 * face));
            d->half_face_bytes = face;
        }
        return LGT_OK;
    }
    static int half_spinor_dslash(lgt_dd* d, int k, int mode) {
        int rc;
        const int n = (int)d->rk.size(), slice = d->V3;
        const size_t face = (size_t)6 * slice * sizeof(T2);
        if ((rc = ensure_half_faces(d)) != LGT_OK) return rc;
        const int dag = mode == 2 ? 1 : 0;
        // faces of every rank's input field, on the main stream (they read the field the previous kernels completed)
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            T2* H = (T2*)d->half_faces[i];
            const int pg = (2 * slice + 127) / 128;
            if (dag) LAUNCH(c, LGT_K_OTHER, (halo_pack_kernel<T, 1>), pg, 128, c->g, (const T2*)fld(c, 7), (const T2*)fld(c, k), H, H + (size_t)6 * slice, slice);
            else LAUNCH(c, LGT_K_OTHER, (halo_pack_kernel<T, 0>), pg, 128, c->g, (const T2*)fld(c, 7), (const T2*)fld(c, k), H, H + (size_t)6 * slice, slice);
        }
        DD_CU(cudaEventRecord(d->ev_ready, d->stream));
        // bulk of every slab on the main stream ...
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const int b0 = c->g.s_begin, e0 = c->g.s_end;
            double* const part0 = c->partials;
            c->g.s_begin = b0 + slice;
            c->g.s_end = e0 - slice;
            c->partials = part0 + slice / 128;
            rc = mode == 1 ? O::dslash(c, fld(c, 7), fld(c, k), fld(c, 3), 0, 1) : O::dslash(c, fld(c, 7), fld(c, k), nullptr, 1, 2, fld(c, 1));
            c->g.s_begin = b0;
            c->g.s_end = e0;
            c->partials = part0;
            if (rc != LGT_OK) return dd_fail(d, rc, c->err.c_str());
        }
        // ... while the faces travel on the halo stream
        DD_CU(cudaStreamWaitEvent(d->halo_stream, d->ev_ready, 0));
        cudaStream_t const main_stream = d->stream;
        d->stream = d->halo_stream;
        const size_t send_off[2] = {0, face}, recv_off[2] = {2 * face, 3 * face};
        rc = dd_exchange_regions(d, d->half_faces.data(), send_off, recv_off, face);
        d->stream = main_stream;
        if (rc != LGT_OK) return rc;
        DD_CU(cudaEventRecord(d->ev_halo, d->halo_stream));
        DD_CU(cudaStreamWaitEvent(d->stream, d->ev_halo, 0));
        // the two boundary slices from the received faces
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const int b0 = c->g.s_begin, e0 = c->g.s_end;
            double* const part0 = c->partials;
            const T2* H = (const T2*)d->half_faces[i];
            const T2 *hi_in = H + (size_t)12 * slice, *lo_in = H + (size_t)18 * slice;
            const T kap = (T)c->kappa;
            const int bg = slice / 128;
            c->g.s_end = b0 + slice;  // first slice: backward t hop from lo_in
            if (mode == 1)
                LAUNCH(c, LGT_K_DSLASH, (dslash_halo_kernel<T, 0, 1, 1>), bg, 128, c->g, (const T2*)fld(c, 7), (const T2*)fld(c, k), (T2*)fld(c, 3), kap,
                       c->st, c->partials, (T2*)nullptr, lo_in, hi_in, b0, e0 - slice);
            else
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_halo_kernel<T, 1, 2, 1>), bg, 128, c->g, (const T2*)fld(c, 7), (const T2*)fld(c, k), (T2*)nullptr, kap,
                       c->st, c->partials, (T2*)fld(c, 1), lo_in, hi_in, b0, e0 - slice);
            c->g.s_begin = e0 - slice;  // last slice: forward t hop from hi_in
            c->g.s_end = e0;
            c->partials = part0 + (e0 - slice - b0) / 128;
            if (mode == 1)
                LAUNCH(c, LGT_K_DSLASH, (dslash_halo_kernel<T, 0, 1, 2>), bg, 128, c->g, (const T2*)fld(c, 7), (const T2*)fld(c, k), (T2*)fld(c, 3), kap,
                       c->st, c->partials, (T2*)nullptr, lo_in, hi_in, b0, e0 - slice);
            else
                LAUNCH(c, LGT_K_DSLASH_R, (dslash_halo_kernel<T, 1, 2, 2>), bg, 128, c->g, (const T2*)fld(c, 7), (const T2*)fld(c, k), (T2*)nullptr, kap,
                       c->st, c->partials, (T2*)fld(c, 1), lo_in, hi_in, b0, e0 - slice);
            c->g.s_begin = b0;
            c->g.s_end = e0;
            c->partials = part0;
        }
        return LGT_OK;
    }
    template <class Launch> static int overlapped(lgt_dd* d, int k, Launch launch) {
        int rc;
        if (!d->halo_stream) {
            DD_CU(cudaStreamCreateWithFlags(&d->halo_stream, cudaStreamNonBlocking));
            DD_CU(cudaEventCreateWithFlags(&d->ev_ready, cudaEventDisableTiming));
            DD_CU(cudaEventCreateWithFlags(&d->ev_halo, cudaEventDisableTiming));
        }
        const int slice = d->V3, n = (int)d->rk.size();
        DD_CU(cudaEventRecord(d->ev_ready, d->stream));  // the field is complete
        for (int i = 0; i < n; i++) {                    // bulk: local slices 2 .. Lt_loc - 1
            lgt_ctx* c = d->rk[i];
            const int b0 = c->g.s_begin, e0 = c->g.s_end;
            double* const part0 = c->partials;
            c->g.s_begin = b0 + slice;
            c->g.s_end = e0 - slice;
            c->partials = part0 + slice / 128;
            rc = launch(c);
            c->g.s_begin = b0;
            c->g.s_end = e0;
            c->partials = part0;
            if (rc != LGT_OK) return dd_fail(d, rc, c->err.c_str());
        }
        DD_CU(cudaStreamWaitEvent(d->halo_stream, d->ev_ready, 0));
        cudaStream_t const main_stream = d->stream;
        d->stream = d->halo_stream;  // dd_exchange enqueues (and, for the host transport, waits) on d->stream
        rc = exchange_spinor(d, k);
        d->stream = main_stream;
        if (rc != LGT_OK) return rc;
        DD_CU(cudaEventRecord(d->ev_halo, d->halo_stream));
        DD_CU(cudaStreamWaitEvent(d->stream, d->ev_halo, 0));
        for (int i = 0; i < n; i++) {  // the two boundary slices
            lgt_ctx* c = d->rk[i];
            const int b0 = c->g.s_begin, e0 = c->g.s_end;
            double* const part0 = c->partials;
            c->g.s_end = b0 + slice;
            rc = launch(c);
            if (rc == LGT_OK) {
                c->g.s_begin = e0 - slice;
                c->g.s_end = e0;
                c->partials = part0 + (e0 - slice - b0) / 128;
                rc = launch(c);
            }
            c->g.s_begin = b0;
            c->g.s_end = e0;
            c->partials = part0;
            if (rc != LGT_OK) return dd_fail(d, rc, c->err.c_str());
        }
        return LGT_OK;
    }

    // Thin-link ghosts current, then the fermions' links c->Uf of every rank: the thin links, or the stout levels built
    // in lockstep with a halo exchange of each level's result (the next level's staples reach into the ghost slices).
    static int fermion_links(lgt_dd* d) {
        int rc;
        if ((rc = dd_exchange_links(d)) != LGT_OK) return rc;
        const int nsm = d->rk[0]->nsmear;
        bool valid = true;
        for (size_t i = 0; i < d->rk.size(); i++) {
            DD_RK(i, O::ensure_fermion_links(d->rk[i]));  // allocation and c->Uf; computes nothing on a slab
            valid = valid && d->rk[i]->usm_valid;
        }
        if (nsm == 0 || valid) return LGT_OK;
        for (int k = 0; k < nsm; k++) {
            std::vector<void*> u;
            for (size_t i = 0; i < d->rk.size(); i++) {
                DD_RK(i, O::smear_level(d->rk[i], k));
                u.push_back(d->rk[i]->Usm[k]);
            }
            if ((rc = dd_exchange(d, u.data(), 36, sizeof(T2))) != LGT_OK) return rc;
        }
        for (lgt_ctx* c : d->rk) c->usm_valid = true;
        return LGT_OK;
    }
    // Pi -= eps F^f from X = ws[0], Y = ws[3] (ghost slices current): the fused kernel, or with smearing the force with
    // respect to U^(n) pulled back level by level as in Ops::fermion_force, G's ghost slices exchanged before each chain
    static int fermion_force(lgt_dd* d, double eps) {
        int rc;
        const int nsm = d->rk[0]->nsmear;
        if (nsm == 0) {
            for (size_t i = 0; i < d->rk.size(); i++) DD_RK(i, O::fermion_force(d->rk[i], d->rk[i]->ws[0], d->rk[i]->ws[3], d->rk[i]->P, 1, eps));
            return LGT_OK;
        }
        const size_t nr = d->rk.size();
        std::vector<T2*> Fa(nr), Fb(nr);
        for (size_t i = 0; i < nr; i++) {
            lgt_ctx* c = d->rk[i];
            if (!c->F2) {
                DD_CU(cudaMalloc(&c->F2, mom_bytes(c)));
                DD_CU(cudaMalloc(&c->F3, mom_bytes(c)));
                DD_CU(cudaMalloc(&c->F4, mom_bytes(c)));
                DD_CU(cudaMemsetAsync(c->F2, 0, mom_bytes(c), d->stream));
                DD_CU(cudaMemsetAsync(c->F3, 0, mom_bytes(c), d->stream));
                DD_CU(cudaMemsetAsync(c->F4, 0, mom_bytes(c), d->stream));
            }
            Fa[i] = (T2*)c->F3;
            Fb[i] = (T2*)c->F4;
            LAUNCH(c, LGT_K_FERMION_FORCE, (fermion_force_kernel<T, 0>), site_blocks(c, 128), 128, c->g, (const T2*)c->Uf, (const T2*)c->ws[0],
                   (const T2*)c->ws[3], Fa[i], (T)c->kappa, (T)0);
        }
        for (int k = nsm - 1; k >= 0; k--) {
            std::vector<void*> g;
            for (size_t i = 0; i < nr; i++) {
                lgt_ctx* c = d->rk[i];
                LAUNCH(c, LGT_K_FERMION_FORCE, (stout_local_kernel<T>), site_blocks(c, 32), 128, c->g, (const T2*)c->Asm[k], Fa[i], (T2*)c->F2);
                g.push_back(c->F2);
            }
            if ((rc = dd_exchange(d, g.data(), 16, sizeof(T2))) != LGT_OK) return rc;
            for (size_t i = 0; i < nr; i++) {
                lgt_ctx* c = d->rk[i];
                const T2* Uk = (const T2*)(k == 0 ? c->U : c->Usm[k - 1]);
                if (k == 0)
                    LAUNCH(c, LGT_K_FERMION_FORCE, (stout_chain_kernel<T, 1>), site_blocks(c, 32), 128, c->g, Uk, (const T2*)c->F2, (const T2*)Fa[i],
                           (T2*)c->P, (T)c->rho, (T)eps);
                else
                    LAUNCH(c, LGT_K_FERMION_FORCE, (stout_chain_kernel<T, 0>), site_blocks(c, 32), 128, c->g, Uk, (const T2*)c->F2, (const T2*)Fa[i],
                           Fb[i], (T)c->rho, (T)0);
                T2* t = Fa[i];
                Fa[i] = Fb[i];
                Fb[i] = t;
            }
        }
        return LGT_OK;
    }

    // out = D in (or D^dag in) on the fields ws[in], ws[out] of every rank
    static int dslash(lgt_dd* d, int in, int out, int dagger) {
        int rc;
        if ((rc = fermion_links(d)) != LGT_OK) return rc;
        if ((rc = exchange_spinor(d, in)) != LGT_OK) return rc;
        for (size_t i = 0; i < d->rk.size(); i++) {
            lgt_ctx* c = d->rk[i];
            DD_RK(i, O::dslash(c, fld(c, 7), fld(c, in), fld(c, out), dagger, 0));
        }
        return LGT_OK;
    }

    // CG on D^dag D, b = ws[ib] (or phi for ib == 6), x = ws[0], workspaces r, p, t = ws[1..3]; leaves Y = D x in ws[3]
    // if want_y.  Same recurrence, stop rule and fused kernels as Ops::cg; every sum is all-reduced over the ranks.
    // pcoef != 0: p = b + pcoef p at the start (the mixed driver's reliable update, as Ops::cg; with pushed halos the ghost
    // slices of p are set from b, so the solve restarts there)
    static int cg(lgt_dd* d, int ib, bool want_y, double tol, int max_iter, int* iters, double* rel, double pcoef = 0.0) {
        int rc;
        if (d->halo_mode == LGT_DD_PUSH) pcoef = 0.0;
        if (!fp32_on_f64(d->rk[0]) && (rc = fermion_links(d)) != LGT_OK) return rc;  // (the mixed driver has done it in fp64)
        const int n = (int)d->rk.size();
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t off = spinor_off(c), cnt = spinor_n(c);
            const T2* b = (const T2*)fld(c, ib) + off;
            LAUNCH(c, LGT_K_CG_BLAS, (cg_init_kernel<T>), stream_blocks(c, cnt), 256, cnt, b, (T2*)fld(c, 0) + off, (T2*)fld(c, 1) + off,
                   (T2*)fld(c, 2) + off, c->st, tol * tol, max_iter, c->partials, c->counter, zmask(c), (T)pcoef);
            LAUNCH(c, LGT_K_CG_BLAS, cg_rr_to_tmp_kernel, 1, 1, c->st);
        }
        if ((rc = allreduce_tmp(d)) != LGT_OK) return rc;
        for (int i = 0; i < n; i++) LAUNCH(d->rk[i], LGT_K_CG_BLAS, (cg_apply_kernel<0>), 1, 1, d->rk[i]->st);
        // pushed halos need the neighbours' buffers of THIS precision: always there for local neighbours, mapped through
        // IPC only for the handle's own precision
        const bool push = d->halo_mode == LGT_DD_PUSH && d->V3 % 128 == 0 && (d->rk.size() == (size_t)d->nranks || !fp32_on_f64(d->rk[0]));
        // LGT_DD_OVERLAP: time slabs of at least three slices whose slices are whole 128-site chunks; else plain exchange
        const bool overlap = d->halo_mode == LGT_DD_OVERLAP && d->Pz == 0 && d->V3 % 128 == 0 && d->Lt_loc >= 3;
        // LGT_DD_HALF: the overlapped schedule with half spinors on the wire; the thin links (no smearing) must be the operator's
        const bool half = d->halo_mode == LGT_DD_HALF && d->Pz == 0 && d->V3 % 128 == 0 && d->Lt_loc >= 3;
        std::vector<Neighbours<T>> push_t(n), push_r(n);
        if (push) {
            // r = p = b on the ghost slices too (one ordinary exchange of b); from here on p's ghosts follow by local
            // arithmetic and the ghosts of t and r are written by the neighbours' Dslash kernels
            if ((rc = exchange_spinor(d, ib)) != LGT_OK) return rc;
            const size_t slice = (size_t)12 * d->V3, hi = (size_t)(d->Lt_loc + 1) * slice;
            for (int i = 0; i < n; i++) {
                lgt_ctx* c = d->rk[i];
                const T2* b = (const T2*)fld(c, ib);
                for (int f = 1; f <= 2; f++) {
                    DD_CU(cudaMemcpyAsync((T2*)fld(c, f), b, slice * sizeof(T2), cudaMemcpyDeviceToDevice, d->stream));
                    DD_CU(cudaMemcpyAsync((T2*)fld(c, f) + hi, b + hi, slice * sizeof(T2), cudaMemcpyDeviceToDevice, d->stream));
                }
                const int r = d->rank_of[i];
                const int dn = dd_local_index(d, (r + d->nranks - 1) % d->nranks), up = dd_local_index(d, (r + 1) % d->nranks);
                push_r[i].lo = (T2*)(dn >= 0 ? fld(d->rk[dn], 1) : d->ipc_peer[0][0]);
                push_r[i].hi = (T2*)(up >= 0 ? fld(d->rk[up], 1) : d->ipc_peer[0][1]);
                push_t[i].lo = (T2*)(dn >= 0 ? fld(d->rk[dn], 3) : d->ipc_peer[1][0]);
                push_t[i].hi = (T2*)(up >= 0 ? fld(d->rk[up], 3) : d->ipc_peer[1][1]);
                if (!push_r[i].lo || !push_r[i].hi || !push_t[i].lo || !push_t[i].hi)
                    return dd_fail(d, LGT_ESTATE, "LGT_DD_PUSH: the neighbours' buffers are not mapped (lgt_dd_ipc_import)");
            }
        }
        lgt_ctx* c0 = d->rk[0];
        int launched = 0;
        for (;;) {
            DD_CU(cudaMemcpyAsync(c0->h_st, c0->st, sizeof(CgState), cudaMemcpyDeviceToHost, d->stream));
            DD_CU(cudaStreamSynchronize(d->stream));
            if (c0->h_st->done) break;
            int chunk = max_iter - launched;
            if (chunk > 8) chunk = 8;
            if (chunk <= 0) chunk = 1;
            for (int it = 0; it < chunk; it++) {
                if (half) {
                    if ((rc = half_spinor_dslash(d, 2, 1)) != LGT_OK) return rc;
                } else if (overlap) {
                    if ((rc = overlapped(d, 2, [&](lgt_ctx* c) { return O::dslash(c, fld(c, 7), fld(c, 2), fld(c, 3), 0, 1); })) != LGT_OK) return rc;
                } else if (!push && (rc = exchange_spinor(d, 2)) != LGT_OK) return rc;  // p
                for (int i = 0; i < n; i++) {
                    lgt_ctx* c = d->rk[i];
                    if (push) DD_RK(i, dslash_pushing(d, c, fld(c, 2), fld(c, 3), 0, 1, nullptr, push_t[i]));
                    else if (!overlap && !half) DD_RK(i, O::dslash(c, fld(c, 7), fld(c, 2), fld(c, 3), 0, 1));  // t = D p, partials of |t|^2
                    LAUNCH(c, LGT_K_CG_BLAS, cg_partial_sum_kernel, 1, 1024, site_blocks(c, 128), c->partials, c->st);
                }
                if ((rc = allreduce_tmp(d)) != LGT_OK) return rc;
                for (int i = 0; i < n; i++) LAUNCH(d->rk[i], LGT_K_CG_BLAS, (cg_apply_kernel<1>), 1, 1, d->rk[i]->st);
                if (half) {
                    if ((rc = half_spinor_dslash(d, 3, 2)) != LGT_OK) return rc;
                } else if (overlap) {
                    if ((rc = overlapped(d, 3, [&](lgt_ctx* c) { return O::dslash(c, fld(c, 7), fld(c, 3), nullptr, 1, 2, fld(c, 1)); })) != LGT_OK)
                        return rc;
                } else if (!push && (rc = exchange_spinor(d, 3)) != LGT_OK) return rc;  // t
                for (int i = 0; i < n; i++) {
                    lgt_ctx* c = d->rk[i];
                    if (push) DD_RK(i, dslash_pushing(d, c, fld(c, 3), nullptr, 1, 2, fld(c, 1), push_r[i]));
                    else if (!overlap && !half) DD_RK(i, O::dslash(c, fld(c, 7), fld(c, 3), nullptr, 1, 2, fld(c, 1)));  // r -= alpha D^dag t, partials of |r|^2
                    LAUNCH(c, LGT_K_CG_BLAS, cg_partial_sum_kernel, 1, 1024, site_blocks(c, 128), c->partials, c->st);
                }
                if ((rc = allreduce_tmp(d)) != LGT_OK) return rc;
                for (int i = 0; i < n; i++) {
                    lgt_ctx* c = d->rk[i];
                    const size_t off = spinor_off(c), cnt = spinor_n(c);
                    LAUNCH(c, LGT_K_CG_BLAS, (cg_apply_kernel<2>), 1, 1, c->st);
                    LAUNCH(c, LGT_K_CG_UPDATE, (cg_update_xp_kernel<T>), stream_blocks(c, cnt), 256, cnt, (T2*)fld(c, 0) + off, (T2*)fld(c, 2) + off,
                           (const T2*)fld(c, 1) + off, c->st);
                    if (push) {
                        const size_t slice = (size_t)12 * d->V3;
                        LAUNCH(c, LGT_K_CG_BLAS, (cg_update_p_ghost_kernel<T>), stream_blocks(c, 2 * slice), 256, slice,
                               (size_t)(d->Lt_loc + 1) * slice, (T2*)fld(c, 2), (const T2*)fld(c, 1), c->st);
                    }
                }
            }
            launched += chunk;
        }
        const CgState& h = *c0->h_st;
        if (iters) *iters = h.iter;
        if (rel) *rel = (h.bb > 0.0) ? sqrt(h.rr / h.bb) : 0.0;
        if (want_y && (rc = dslash(d, 0, 3, 0)) != LGT_OK) return rc;
        if (h.rr > h.tol2 * h.bb) return dd_fail(d, LGT_ENOCONV, "CG did not reach the tolerance within max_iter");
        return LGT_OK;
    }

    // Pi -= eps F^g on every rank
    static int kick_gauge(lgt_dd* d, double eps) {
        int rc;
        if ((rc = dd_exchange_links(d)) != LGT_OK) return rc;
        for (size_t i = 0; i < d->rk.size(); i++) DD_RK(i, O::gauge_force(d->rk[i], d->rk[i]->P, 1, eps));
        return LGT_OK;
    }
    // Pi -= eps F^f on every rank (solve, halo of X and Y, force kernels); nothing without fermions
    static int kick_fermion(lgt_dd* d, double eps, double tol, int max_iter, int* cg_iters) {
        int rc, it = 0, conv = LGT_OK;
        if (fermions_on(d->rk[0])) {
            rc = d->rk[0]->action == LGT_ACTION_EO ? eo_solve(d, true, tol, max_iter, &it, false) : dd_solve(d, 6, true, tol, max_iter, &it);
            if (rc == LGT_ENOCONV) conv = rc;
            else if (rc != LGT_OK) return rc;
            if ((rc = exchange_spinor(d, 0)) != LGT_OK) return rc;  // X(x + mu)
            if ((rc = exchange_spinor(d, 3)) != LGT_OK) return rc;  // Y(x + mu)
            if ((rc = fermion_force(d, eps)) != LGT_OK) return rc;
        }
        if (cg_iters) *cg_iters = it;
        return conv;
    }
    // Pi -= eps (F^g + F^f) on every rank
    static int kick(lgt_dd* d, double eps, double tol, int max_iter, int* cg_iters) {
        int rc;
        if ((rc = kick_gauge(d, eps)) != LGT_OK) return rc;
        return kick_fermion(d, eps, tol, max_iter, cg_iters);
    }

    static int drift(lgt_dd* d, double eps) {
        for (size_t i = 0; i < d->rk.size(); i++) DD_RK(i, O::link_update(d->rk[i], eps));
        d->links_ghost_valid = false;
        return dd_exchange_links(d);
    }

    // S_g, S_F, K summed over the ranks (device slots scal[0..2] of every rank, one all-reduce of three doubles)
    // eta_norm: S_F = |eta|^2 of the heat-bath field in ws[4] instead of a solve (the start of an HMC trajectory)
    static int action(lgt_dd* d, double tol, int max_iter, double* S_g, double* S_F, double* K, int* cg_iters, bool eta_norm = false) {
        int rc, it = 0, conv = LGT_OK;
        if ((rc = dd_exchange_links(d)) != LGT_OK) return rc;
        const bool ferm = fermions_on(d->rk[0]) && S_F != nullptr;
        const bool eo = d->rk[0]->action == LGT_ACTION_EO;
        if (ferm && !eta_norm) {
            rc = eo ? eo_solve(d, false, tol, max_iter, &it, true) : dd_solve(d, 6, false, tol, max_iter, &it);
            if (rc == LGT_ENOCONV) conv = rc;
            else if (rc != LGT_OK) return rc;
        }
        std::vector<double*> slots;
        for (size_t i = 0; i < d->rk.size(); i++) {
            lgt_ctx* c = d->rk[i];
            DD_RK(i, O::plaquette_sum(c, c->scal + 0));
            DD_RK(i, O::kinetic(c, c->scal + 1));
            if (ferm && eo) {
                if (eta_norm) {  // |eta_e|^2; after a solve eo_solve() has left Re <phi_e, X_e> in the slot already
                    const size_t off = half_off(c), cnt = half_n(c);
                    LAUNCH(c, LGT_K_OTHER, (redot_kernel<T>), stream_blocks(c, cnt), 256, cnt, (const T2*)hB(c) + off, (const T2*)hB(c) + off,
                           c->scal + 2, c->partials, c->counter, zmask_half(c));
                }
            } else if (ferm) {
                const size_t off = spinor_off(c);
                const T2 *a = (const T2*)(eta_norm ? c->ws[4] : c->phi) + off, *b = (const T2*)(eta_norm ? c->ws[4] : c->ws[0]) + off;
                LAUNCH(c, LGT_K_OTHER, (redot_kernel<T>), stream_blocks(c, spinor_n(c)), 256, spinor_n(c), a, b, c->scal + 2, c->partials, c->counter,
                       zmask(c));
            } else {
                DD_CU(cudaMemsetAsync(c->scal + 2, 0, sizeof(double), d->stream));
            }
            slots.push_back(c->scal);
        }
        if ((rc = dd_allreduce(d, slots.data(), 3)) != LGT_OK) return rc;
        lgt_ctx* c0 = d->rk[0];
        DD_CU(cudaMemcpyAsync(c0->h_scal, c0->scal, 3 * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
        DD_CU(cudaStreamSynchronize(d->stream));
        const double sites = d->Pz > 0 ? (double)d->Vglob : (double)d->V3 * d->Lt_loc * d->nranks;
        if (S_g) *S_g = c0->beta * (6.0 * sites - c0->h_scal[0]);
        if (K) *K = c0->h_scal[1];
        if (S_F) *S_F = ferm ? c0->h_scal[2] : 0.0;
        if (cg_iters) *cg_iters = it;
        return conv;
    }

    // ---- even/odd preconditioned action on the slabs.  A rank's LOCAL parity (x + y + z + t_local) differs from the global
    // one by t_off, so the globally even sites are the local parity pe = t_off & 1; everything else is Ops<T>'s even/odd
    // code with (pe, 1 - pe) in place of (0, 1), the input half field's ghost slices exchanged before every hop and the
    // CG sums all-reduced.  Half fields have V3 / 2 sites per time slice, so their slices are contiguous runs too.
    static int pe_of(const lgt_ctx* c) { return (c->g.t_off + c->g.z_off) & 1; }  // z_off = 0 on time slabs
    static T2* E(lgt_ctx* c, int k) { return O::eo_field(c, k + pe_of(c)); }      // globally even member of the pair (k, k+1)
    static T2* Od(lgt_ctx* c, int k) { return O::eo_field(c, k + 1 - pe_of(c)); }  // globally odd member
    typedef T2* (*HalfSel)(lgt_ctx*);
    static int exchange_half(lgt_dd* d, HalfSel sel) {
        std::vector<void*> f;
        for (lgt_ctx* c : d->rk) f.push_back(sel(c));
        return dd_exchange(d, f.data(), 6, sizeof(T2));  // 12 components x V3 / 2 sites per slice
    }
    static T2* hXe(lgt_ctx* c) { return E(c, 0); }
    static T2* hXo(lgt_ctx* c) { return Od(c, 0); }
    static T2* hYe(lgt_ctx* c) { return E(c, 2); }
    static T2* hP(lgt_ctx* c) { return O::eo_field(c, 6); }
    static T2* hT(lgt_ctx* c) { return O::eo_field(c, 7); }
    // the streaming sums over a half field of a grid rank: an xy plane holds L0 L1 / 2 half-field sites
    static ZMask zmask_half(const lgt_ctx* c) {
        ZMask m = zmask(c);
        m.xy >>= 1;
        return m;
    }
    static size_t half_off(const lgt_ctx* c) { return (size_t)12 * c->g.h_begin; }
    static size_t half_n(const lgt_ctx* c) { return (size_t)12 * (c->g.h_end - c->g.h_begin); }
    // one hop on every rank, after the exchange of its input field
    // push: the result's boundary slices are stored into the neighbours' ghost slices by the kernel (modes 1, 2);
    // input_current: the input's ghost slices are already up to date (pushed, or maintained locally), no exchange
    static int hop_all(lgt_dd* d, bool to_even, HalfSel in, HalfSel self, HalfSel out, int dagger, int mode, bool plus_kappa, HalfSel r = nullptr,
                       const std::vector<Neighbours<T>>* push = nullptr, bool input_current = false) {
        int rc;
        // LGT_DD_OVERLAP (and LGT_DD_HALF, which has no half-field form): the exchange of the input half field on the halo
        // stream under the bulk of the slab, the two boundary slices after it -- DdOps::overlapped for the half-field range.
        // Block partials land where a single launch would put them: in fp64 bitwise the iterates of LGT_DD_EXCHANGE.
        const int hslice = d->V3 / 2;
        // LGT_DD_HALF: the same schedule with half spinors on the wire (halo_pack_cb_kernel / hop_cb_halo_kernel; modes 0 - 3)
        if (!input_current && !push && d->halo_mode == LGT_DD_HALF && d->Pz == 0 && hslice % 128 == 0 && d->Lt_loc >= 3) {
            if ((rc = ensure_half_faces(d)) != LGT_OK) return rc;
            const size_t face = (size_t)6 * hslice * sizeof(T2);
            const int n = (int)d->rk.size();
            for (int i = 0; i < n; i++) {  // faces of the input field, on the main stream
                lgt_ctx* c = d->rk[i];
                const int p = to_even ? pe_of(c) : 1 - pe_of(c);
                T2* H = (T2*)d->half_faces[i];
                const int pg = (2 * hslice + 127) / 128;
                if (dagger) LAUNCH(c, LGT_K_OTHER, (halo_pack_cb_kernel<T, 1>), pg, 128, c->g, O::links_cb(c, 1 - p), (const T2*)in(c), H, H + (size_t)6 * hslice, hslice);
                else LAUNCH(c, LGT_K_OTHER, (halo_pack_cb_kernel<T, 0>), pg, 128, c->g, O::links_cb(c, 1 - p), (const T2*)in(c), H, H + (size_t)6 * hslice, hslice);
            }
            DD_CU(cudaEventRecord(d->ev_ready, d->stream));
            for (int i = 0; i < n; i++) {  // bulk
                lgt_ctx* c = d->rk[i];
                const int p = to_even ? pe_of(c) : 1 - pe_of(c);
                const double kap = plus_kappa ? c->kappa : -c->kappa;
                const int b0 = c->g.h_begin, e0 = c->g.h_end;
                double* const part0 = c->partials;
                c->g.h_begin = b0 + hslice;
                c->g.h_end = e0 - hslice;
                c->partials = part0 + hslice / 128;
                rc = O::hop(c, p, in(c), self ? self(c) : nullptr, out ? out(c) : nullptr, dagger, mode, kap, r ? r(c) : nullptr);
                c->g.h_begin = b0;
                c->g.h_end = e0;
                c->partials = part0;
                if (rc != LGT_OK) return dd_fail(d, rc, c->err.c_str());
            }
            DD_CU(cudaStreamWaitEvent(d->halo_stream, d->ev_ready, 0));
            cudaStream_t const main_stream = d->stream;
            d->stream = d->halo_stream;
            const size_t send_off[2] = {0, face}, recv_off[2] = {2 * face, 3 * face};
            rc = dd_exchange_regions(d, d->half_faces.data(), send_off, recv_off, face);
            d->stream = main_stream;
            if (rc != LGT_OK) return rc;
            DD_CU(cudaEventRecord(d->ev_halo, d->halo_stream));
            DD_CU(cudaStreamWaitEvent(d->stream, d->ev_halo, 0));
            for (int i = 0; i < n; i++) {  // the two boundary slices from the received faces
                lgt_ctx* c = d->rk[i];
                const int p = to_even ? pe_of(c) : 1 - pe_of(c);
                const T kap = (T)(plus_kappa ? c->kappa : -c->kappa);
                const int b0 = c->g.h_begin, e0 = c->g.h_end;
                double* const part0 = c->partials;
                const T2* H = (const T2*)d->half_faces[i];
                const T2 *hi_in = H + (size_t)12 * hslice, *lo_in = H + (size_t)18 * hslice;
                const int bg = hslice / 128;
                const T2 *Up = O::links_cb(c, p), *Uq = O::links_cb(c, 1 - p);
                const T2* sf = self ? (const T2*)self(c) : nullptr;
                T2* of = out ? out(c) : nullptr;
                T2* rf = r ? r(c) : nullptr;
                rc = LGT_OK;
                for (int side = 0; side < 2 && rc == LGT_OK; side++) {
                    if (side == 0) {
                        c->g.h_begin = b0;
                        c->g.h_end = b0 + hslice;
                        c->partials = part0;
                    } else {
                        c->g.h_begin = e0 - hslice;
                        c->g.h_end = e0;
                        c->partials = part0 + (e0 - hslice - b0) / 128;
                    }
                    rc = [&]() -> int {
#define HALO_ARGS c->g, p, Up, Uq, (const T2*)in(c), sf, of, kap, c->st, c->partials, rf, lo_in, hi_in
#define HALO_LAUNCH(DAG, MODE, KC)                                                                                   \
    do {                                                                                                             \
        if (side == 0) LAUNCH(c, KC, (hop_cb_halo_kernel<T, DAG, MODE, 1>), bg, 128, HALO_ARGS);                     \
        else LAUNCH(c, KC, (hop_cb_halo_kernel<T, DAG, MODE, 2>), bg, 128, HALO_ARGS);                               \
    } while (0)
                        if (mode == 0 && !dagger) HALO_LAUNCH(0, 0, LGT_K_DSLASH);
                        else if (mode == 0) HALO_LAUNCH(1, 0, LGT_K_DSLASH);
                        else if (mode == 3 && !dagger) HALO_LAUNCH(0, 3, LGT_K_DSLASH);
                        else if (mode == 3) HALO_LAUNCH(1, 3, LGT_K_DSLASH);
                        else if (mode == 1) HALO_LAUNCH(0, 1, LGT_K_DSLASH);
                        else HALO_LAUNCH(1, 2, LGT_K_DSLASH_R);
#undef HALO_LAUNCH
#undef HALO_ARGS
                        return LGT_OK;
                    }();
                }
                c->g.h_begin = b0;
                c->g.h_end = e0;
                c->partials = part0;
                if (rc != LGT_OK) return dd_fail(d, rc, c->err.c_str());
            }
            return LGT_OK;
        }
        if (!input_current && !push && (d->halo_mode == LGT_DD_OVERLAP || d->halo_mode == LGT_DD_HALF) && d->Pz == 0 && hslice % 128 == 0 &&
            d->Lt_loc >= 3) {
            if (!d->halo_stream) {
                DD_CU(cudaStreamCreateWithFlags(&d->halo_stream, cudaStreamNonBlocking));
                DD_CU(cudaEventCreateWithFlags(&d->ev_ready, cudaEventDisableTiming));
                DD_CU(cudaEventCreateWithFlags(&d->ev_halo, cudaEventDisableTiming));
            }
            auto launch = [&](lgt_ctx* c) {
                const int p = to_even ? pe_of(c) : 1 - pe_of(c);
                const double kap = plus_kappa ? c->kappa : -c->kappa;
                return O::hop(c, p, in(c), self ? self(c) : nullptr, out ? out(c) : nullptr, dagger, mode, kap, r ? r(c) : nullptr);
            };
            DD_CU(cudaEventRecord(d->ev_ready, d->stream));  // the input field is complete
            for (size_t i = 0; i < d->rk.size(); i++) {      // bulk: the slices that touch no ghost slice
                lgt_ctx* c = d->rk[i];
                const int b0 = c->g.h_begin, e0 = c->g.h_end;
                double* const part0 = c->partials;
                c->g.h_begin = b0 + hslice;
                c->g.h_end = e0 - hslice;
                c->partials = part0 + hslice / 128;
                rc = launch(c);
                c->g.h_begin = b0;
                c->g.h_end = e0;
                c->partials = part0;
                if (rc != LGT_OK) return dd_fail(d, rc, c->err.c_str());
            }
            DD_CU(cudaStreamWaitEvent(d->halo_stream, d->ev_ready, 0));
            cudaStream_t const main_stream = d->stream;
            d->stream = d->halo_stream;
            rc = exchange_half(d, in);
            d->stream = main_stream;
            if (rc != LGT_OK) return rc;
            DD_CU(cudaEventRecord(d->ev_halo, d->halo_stream));
            DD_CU(cudaStreamWaitEvent(d->stream, d->ev_halo, 0));
            for (size_t i = 0; i < d->rk.size(); i++) {  // the two boundary slices
                lgt_ctx* c = d->rk[i];
                const int b0 = c->g.h_begin, e0 = c->g.h_end;
                double* const part0 = c->partials;
                c->g.h_end = b0 + hslice;
                rc = launch(c);
                if (rc == LGT_OK) {
                    c->g.h_begin = e0 - hslice;
                    c->g.h_end = e0;
                    c->partials = part0 + (e0 - hslice - b0) / 128;
                    rc = launch(c);
                }
                c->g.h_begin = b0;
                c->g.h_end = e0;
                c->partials = part0;
                if (rc != LGT_OK) return dd_fail(d, rc, c->err.c_str());
            }
            return LGT_OK;
        }
        if (!input_current && (rc = exchange_half(d, in)) != LGT_OK) return rc;
        for (size_t i = 0; i < d->rk.size(); i++) {
            lgt_ctx* c = d->rk[i];
            const int p = to_even ? pe_of(c) : 1 - pe_of(c);
            const double kap = plus_kappa ? c->kappa : -c->kappa;
            if (push)
                DD_RK(i, split_launch(c, &c->g.h_begin, &c->g.h_end, d->V3 / 2, d->Lt_loc, (*push)[i], [&](const PushTo<T>* to) {
                          return O::hop(c, p, in(c), self ? self(c) : nullptr, out ? out(c) : nullptr, dagger, mode, kap, r ? r(c) : nullptr, to);
                      }));
            else
                DD_RK(i, O::hop(c, p, in(c), self ? self(c) : nullptr, out ? out(c) : nullptr, dagger, mode, kap, r ? r(c) : nullptr));
        }
        return LGT_OK;
    }
    // where rank i's kernels push the boundary slices of the half field `sel` (neighbours in this process only)
    static bool push_targets(lgt_dd* d, HalfSel sel, std::vector<Neighbours<T>>& to) {
        to.resize(d->rk.size());
        for (size_t i = 0; i < d->rk.size(); i++) {
            const int r = d->rank_of[i];
            const int dn = dd_local_index(d, (r + d->nranks - 1) % d->nranks), up = dd_local_index(d, (r + 1) % d->nranks);
            if (dn < 0 || up < 0) return false;
            to[i].lo = sel(d->rk[dn]);
            to[i].hi = sel(d->rk[up]);
        }
        return true;
    }
    static T2* hB(lgt_ctx* c) { return E(c, 4); }
    static T2* hR(lgt_ctx* c) { return Od(c, 4); }  // the odd half of the split source is free: CG residual

    // X_e = (M^dag M)^-1 phi_e on every rank; then, if want_xy, the full fields X = ws[0], Y = ws[3] of the force kernel
    // the k-th half field of this precision's set (for DdOps<float> on an LGT_F64 group: the fp32 set b, e, r, p, u, t)
    template <int K> static T2* F(lgt_ctx* c) { return O::eo_field(c, K); }
    // CG on M^dag M over the globally even sites of every rank: x = 0 start, the recurrence, stop rule and fused kernels
    // of Ops::eo_cg, input ghost slices exchanged before every hop, sums all-reduced.  B, X, R, P, U: even half fields,
    // Tt: an odd scratch field.  Returns the final recurrence state through *state.
    static int eo_cg_loop(lgt_dd* d, HalfSel B, HalfSel X, HalfSel R, HalfSel P, HalfSel Uu, HalfSel Tt, double tol, int max_iter,
                          CgState* state, double pcoef = 0.0) {
        int rc;
        if (d->halo_mode == LGT_DD_PUSH) pcoef = 0.0;  // as in cg()
        const int n = (int)d->rk.size();
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t off = half_off(c), cnt = half_n(c);
            LAUNCH(c, LGT_K_CG_BLAS, (cg_init_kernel<T>), stream_blocks(c, cnt), 256, cnt, (const T2*)B(c) + off, X(c) + off, R(c) + off,
                   P(c) + off, c->st, tol * tol, max_iter, c->partials, c->counter, zmask_half(c), (T)pcoef);
            LAUNCH(c, LGT_K_CG_BLAS, cg_rr_to_tmp_kernel, 1, 1, c->st);
        }
        if ((rc = allreduce_tmp(d)) != LGT_OK) return rc;
        for (int i = 0; i < n; i++) LAUNCH(d->rk[i], LGT_K_CG_BLAS, (cg_apply_kernel<0>), 1, 1, d->rk[i]->st);
        // LGT_DD_PUSH (neighbours in this process; between processes the half fields are not IPC-mapped and the exchange
        // stays): u and r are pushed by the hops that produce them, each followed by an all-reduce that is the barrier; p's
        // ghost slices follow by local arithmetic; the two odd intermediates t have no collective behind them and are
        // exchanged as before.
        std::vector<Neighbours<T>> push_u, push_r;
        const bool push = d->halo_mode == LGT_DD_PUSH && (d->V3 / 2) % 128 == 0 && push_targets(d, Uu, push_u) && push_targets(d, R, push_r);
        if (push) {
            if ((rc = exchange_half(d, B)) != LGT_OK) return rc;  // r = p = b on the ghost slices too
            const size_t slice = (size_t)6 * d->V3, hi = (size_t)(d->Lt_loc + 1) * slice;
            for (int i = 0; i < n; i++) {
                lgt_ctx* c = d->rk[i];
                for (HalfSel f : {R, P}) {
                    DD_CU(cudaMemcpyAsync(f(c), B(c), slice * sizeof(T2), cudaMemcpyDeviceToDevice, d->stream));
                    DD_CU(cudaMemcpyAsync(f(c) + hi, B(c) + hi, slice * sizeof(T2), cudaMemcpyDeviceToDevice, d->stream));
                }
            }
        }
        lgt_ctx* c0 = d->rk[0];
        int launched = 0;
        auto sum_and = [&](int what) -> int {
            for (int i = 0; i < n; i++) {
                lgt_ctx* c = d->rk[i];
                LAUNCH(c, LGT_K_CG_BLAS, cg_partial_sum_kernel, 1, 1024, (own_half_sites(c) + 127) / 128, c->partials, c->st);
            }
            int r2 = allreduce_tmp(d);
            if (r2 != LGT_OK) return r2;
            for (int i = 0; i < n; i++) {
                if (what == 1) LAUNCH(d->rk[i], LGT_K_CG_BLAS, (cg_apply_kernel<1>), 1, 1, d->rk[i]->st);
                else LAUNCH(d->rk[i], LGT_K_CG_BLAS, (cg_apply_kernel<2>), 1, 1, d->rk[i]->st);
            }
            return LGT_OK;
        };
        for (;;) {
            DD_CU(cudaMemcpyAsync(c0->h_st, c0->st, sizeof(CgState), cudaMemcpyDeviceToHost, d->stream));
            DD_CU(cudaStreamSynchronize(d->stream));
            if (c0->h_st->done) break;
            int chunk = max_iter - launched;
            if (chunk > 8) chunk = 8;
            if (chunk <= 0) chunk = 1;
            for (int it = 0; it < chunk; it++) {
                if ((rc = hop_all(d, false, P, nullptr, Tt, 0, 3, false, nullptr, nullptr, push)) != LGT_OK) return rc;  // t_o = kappa H_oe p
                if ((rc = hop_all(d, true, Tt, P, Uu, 0, 1, true, nullptr, push ? &push_u : nullptr)) != LGT_OK) return rc;  // u = M p, |u|^2
                if ((rc = sum_and(1)) != LGT_OK) return rc;
                if ((rc = hop_all(d, false, Uu, nullptr, Tt, 1, 3, false, nullptr, nullptr, push)) != LGT_OK) return rc;  // t_o = kappa H_oe^dag u
                if ((rc = hop_all(d, true, Tt, Uu, nullptr, 1, 2, true, R, push ? &push_r : nullptr)) != LGT_OK) return rc;  // r -= alpha M^dag u
                if ((rc = sum_and(2)) != LGT_OK) return rc;
                for (int i = 0; i < n; i++) {
                    lgt_ctx* c = d->rk[i];
                    const size_t off = half_off(c), cnt = half_n(c);
                    LAUNCH(c, LGT_K_CG_UPDATE, (cg_update_xp_kernel<T>), stream_blocks(c, cnt), 256, cnt, X(c) + off, P(c) + off,
                           (const T2*)R(c) + off, c->st);
                    if (push) {
                        const size_t slice = (size_t)6 * d->V3;
                        LAUNCH(c, LGT_K_CG_BLAS, (cg_update_p_ghost_kernel<T>), stream_blocks(c, 2 * slice), 256, slice,
                               (size_t)(d->Lt_loc + 1) * slice, P(c), (const T2*)R(c), c->st);
                    }
                }
            }
            launched += chunk;
        }
        *state = *c0->h_st;
        return LGT_OK;
    }

    // X_e = (M^dag M)^-1 phi_e on every rank; then, if want_xy, the full fields X = ws[0], Y = ws[3] of the force kernel
    static int eo_solve(lgt_dd* d, bool want_xy, double tol, int max_iter, int* iters, bool sf_to_slot2) {
        int rc;
        if ((rc = fermion_links(d)) != LGT_OK) return rc;
        const int n = (int)d->rk.size();
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            DD_RK(i, O::eo_ensure(c));
            DD_RK(i, O::eo_split(c, c->phi, O::eo_field(c, 4)));
        }
        CgState h;
        memset(&h, 0, sizeof h);
        bool converged = true;
        if (d->prec == LGT_F64 && sizeof(T) == 8 && d->rk[0]->solver == LGT_SOLVER_MIXED_CG) {
            rc = dd_eo_cg_mixed(d, tol, max_iter, &h.iter);
            if (rc == LGT_ENOCONV) converged = false;
            else if (rc != LGT_OK) return rc;
        } else {
            if ((rc = eo_cg_loop(d, hB, hXe, hR, hP, hYe, hT, tol, max_iter, &h)) != LGT_OK) return rc;
            converged = !(h.rr > h.tol2 * h.bb);
        }
        if (iters) *iters = h.iter;
        if (sf_to_slot2)
            for (int i = 0; i < n; i++) {
                lgt_ctx* c = d->rk[i];
                const size_t off = half_off(c), cnt = half_n(c);
                LAUNCH(c, LGT_K_OTHER, (redot_kernel<T>), stream_blocks(c, cnt), 256, cnt, (const T2*)hB(c) + off, (const T2*)hXe(c) + off,
                       c->scal + 2, c->partials, c->counter, zmask_half(c));
            }
        if (want_xy) {
            if ((rc = hop_all(d, false, hXe, nullptr, hXo, 0, 0, false)) != LGT_OK) return rc;  // X_o = kappa H_oe X_e
            if ((rc = hop_all(d, true, hXo, hXe, hYe, 0, 0, true)) != LGT_OK) return rc;        // Y_e = M X_e
            if ((rc = hop_all(d, false, hYe, nullptr, [](lgt_ctx* c) { return Od(c, 2); }, 1, 0, false)) != LGT_OK) return rc;  // Y_o
            for (int i = 0; i < n; i++) {
                lgt_ctx* c = d->rk[i];
                DD_RK(i, O::eo_merge(c, O::eo_field(c, 0), c->ws[0]));
                DD_RK(i, O::eo_merge(c, O::eo_field(c, 2), c->ws[3]));
            }
        }
        if (!converged) return dd_fail(d, LGT_ENOCONV, "even/odd CG did not reach the tolerance within max_iter");
        return LGT_OK;
    }

    struct Moves {
        lgt_dd* d;
        double tol;
        int max_iter;
        int kick(double eps, int* it) { return DdOps::kick(d, eps, tol, max_iter, it); }
        int kick_gauge(double eps) { return DdOps::kick_gauge(d, eps); }
        int kick_fermion(double eps, int* it) { return DdOps::kick_fermion(d, eps, tol, max_iter, it); }
        int drift(double eps) { return DdOps::drift(d, eps); }
        int inner_gauge_steps(double h, int m) { return plain_inner_gauge_steps(*this, h, m); }  // exchanges in between: no graph
    };
    static int integrate(lgt_dd* d, int nsteps, double dt, double tol, int max_iter, long* cg_iters) {
        Moves m{d, tol, max_iter};
        return integrate_with(m, d->rk[0]->integrator, d->rk[0]->n_inner, nsteps, dt, cg_iters);
    }

    // Heat baths by global element number (reading A-25), so that the fields are those of the undivided lattice
    static int heatbaths(lgt_dd* d, unsigned long long seed, unsigned traj) {
        int rc;
        for (size_t i = 0; i < d->rk.size(); i++) {
            lgt_ctx* c = d->rk[i];
            DD_RK(i, O::momentum_heatbath(c, seed, traj));
            if (c->kappa != 0.0) {
                LAUNCH(c, LGT_K_OTHER, (spinor_heatbath_kernel<T>), stream_blocks(c, (size_t)12 * c->g.Vs), 256, c->g, (T2*)c->ws[4], seed, traj);
                c->has_phi = true;
            }
        }
        if (d->rk[0]->kappa == 0.0) return LGT_OK;
        if (d->rk[0]->action != LGT_ACTION_EO) return dslash(d, 4, 6, 1);  // phi = D^dag eta
        // even/odd action: phi_e = M^dag eta_e, phi_o = 0; eta_e stays in the even member of fields (4, 5) for |eta_e|^2
        if ((rc = fermion_links(d)) != LGT_OK) return rc;
        for (size_t i = 0; i < d->rk.size(); i++) {
            lgt_ctx* c = d->rk[i];
            DD_RK(i, O::eo_ensure(c));
            DD_RK(i, O::eo_split(c, c->ws[4], O::eo_field(c, 4)));
        }
        if ((rc = hop_all(d, false, hB, nullptr, hT, 1, 0, false)) != LGT_OK) return rc;
        if ((rc = hop_all(d, true, hT, hB, hYe, 1, 0, true)) != LGT_OK) return rc;
        for (size_t i = 0; i < d->rk.size(); i++) {
            lgt_ctx* c = d->rk[i];
            DD_CU(cudaMemsetAsync(Od(c, 2), 0, (size_t)12 * c->g.Vhs * sizeof(T2), d->stream));
            DD_RK(i, O::eo_merge(c, O::eo_field(c, 2), c->phi));
        }
        return LGT_OK;
    }
    static int hmc_trajectory(lgt_dd* d, int nsteps, double dt, double tol, int max_iter, unsigned long long seed, unsigned traj,
                              double* dH, int* accepted, long* cg_iters, double* H_initial) {
        int rc, it = 0, conv = LGT_OK;
        long total = 0;
        double sg, sf, k;
        if ((rc = dd_exchange_links(d)) != LGT_OK) return rc;
        for (size_t i = 0; i < d->rk.size(); i++) {
            lgt_ctx* c = d->rk[i];
            if (!c->Usave) DD_CU(cudaMalloc(&c->Usave, links_bytes(c)));
            DD_CU(cudaMemcpyAsync(c->Usave, c->U, links_bytes(c), cudaMemcpyDeviceToDevice, d->stream));
        }
        if ((rc = heatbaths(d, seed, traj)) != LGT_OK) return rc;
        if ((rc = action(d, tol, max_iter, &sg, &sf, &k, &it, true)) != LGT_OK) return rc;
        const double H0 = k + sg + sf;
        rc = integrate(d, nsteps, dt, tol, max_iter, &total);
        if (rc == LGT_ENOCONV) conv = rc;
        else if (rc != LGT_OK) return rc;
        it = 0;
        rc = action(d, tol, max_iter, &sg, &sf, &k, &it);
        if (rc == LGT_ENOCONV) conv = rc;
        else if (rc != LGT_OK) return rc;
        total += it;
        const double dh = (k + sg + sf) - H0;
        const bool acc = metropolis_uniform(seed, traj) < exp(-dh);  // the same all-reduced numbers on every rank
        if (!acc) {
            for (lgt_ctx* c : d->rk) {
                DD_CU(cudaMemcpyAsync(c->U, c->Usave, links_bytes(c), cudaMemcpyDeviceToDevice, d->stream));
                c->usm_valid = c->u32_valid = c->ucb_valid = c->ucb32_valid = false;
            }
            d->links_ghost_valid = true;  // saved with current ghosts
        }
        DD_CU(cudaStreamSynchronize(d->stream));
        if (dH) *dH = dh;
        if (accepted) *accepted = acc ? 1 : 0;
        if (cg_iters) *cg_iters = total;
        if (H_initial) *H_initial = H0;
        return conv;
    }
};

#define DD_DISPATCH(d, fn, ...) ((d)->prec == LGT_F64 ? DdOps<double>::fn(__VA_ARGS__) : DdOps<float>::fn(__VA_ARGS__))

// Mixed-precision solve on a decomposed lattice: the defect correction of cg_mixed() with every rank's fp32 copies
// (links incl. ghost slices, five spinor buffers) and the decomposed fp32 CG inside; true fp64 residual, all-reduced.
// b = field ib, x = ws[0]; r, q, t = ws[1], ws[2], ws[3]; leaves Y = D x in ws[3].
int dd_cg_mixed(lgt_dd* d, int ib, bool want_y, double tol, int max_iter, int* iters) {
    typedef DdOps<double> D64;
    typedef DdOps<float> D32;
    int rc;
    if ((rc = D64::fermion_links(d)) != LGT_OK) return rc;
    const int n = (int)d->rk.size();
    std::vector<double*> slot;
    for (int i = 0; i < n; i++) {
        lgt_ctx* c = d->rk[i];
        const size_t nfull = (size_t)12 * c->g.Vs, nu = (size_t)36 * c->g.Vs;
        if (!c->U32) {
            DD_CU(cudaMalloc(&c->U32, nu * sizeof(float2)));
            for (int k = 0; k < 5; k++) {
                DD_CU(cudaMalloc(&c->ws32[k], nfull * sizeof(float2)));
                DD_CU(cudaMemsetAsync(c->ws32[k], 0, nfull * sizeof(float2), d->stream));
            }
            c->u32_valid = false;
        }
        if (!c->u32_valid) {  // ghost slices included: the links were exchanged above
            LAUNCH(c, LGT_K_OTHER, down_convert_kernel, stream_blocks(c, nu), 256, nu, (const double2*)c->Uf, (float2*)c->U32, 1.0);
            c->u32_valid = true;
        }
        const size_t off = D64::spinor_off(c), cnt = D64::spinor_n(c);
        const double2* b = (const double2*)D64::fld(c, ib);
        DD_CU(cudaMemsetAsync(c->ws[0], 0, nfull * sizeof(double2), d->stream));
        DD_CU(cudaMemsetAsync(c->ws[3], 0, nfull * sizeof(double2), d->stream));
        DD_CU(cudaMemcpyAsync(c->ws[1], b, nfull * sizeof(double2), cudaMemcpyDeviceToDevice, d->stream));
        LAUNCH(c, LGT_K_OTHER, (redot_kernel<double>), stream_blocks(c, cnt), 256, cnt, b + off, b + off, c->scal + 3, c->partials, c->counter,
               D64::zmask(c));
        slot.push_back(c->scal + 3);
    }
    lgt_ctx* c0 = d->rk[0];
    auto read_sum = [&](double& out) -> int {
        int r2 = dd_allreduce(d, slot.data(), 1);
        if (r2 != LGT_OK) return r2;
        DD_CU(cudaMemcpyAsync(c0->h_scal + 3, c0->scal + 3, sizeof(double), cudaMemcpyDeviceToHost, d->stream));
        DD_CU(cudaStreamSynchronize(d->stream));
        out = c0->h_scal[3];
        return LGT_OK;
    };
    double bb = 0.0;
    if ((rc = read_sum(bb)) != LGT_OK) return rc;
    double rr = bb;
    int total = 0, outer = 0, conv = LGT_OK, prev_it = 0;
    double prev_scale = 1.0;
    bool prev_good = false;
    while (bb > 0.0 && rr > tol * tol * bb) {
        if (total >= max_iter || outer >= 40) {
            conv = LGT_ENOCONV;
            break;
        }
        const double scale = 1.0 / sqrt(rr);
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t nfull = (size_t)12 * c->g.Vs;
            LAUNCH(c, LGT_K_CG_BLAS, down_convert_kernel, stream_blocks(c, nfull), 256, nfull, (const double2*)c->ws[1], (float2*)c->ws32[0], scale);
        }
        double eps = 0.25 * tol * sqrt(bb / rr);
        if (eps < c0->inner_tol) eps = c0->inner_tol;
        double pcoef = 0.0;  // reliable update instead of a restart, as in cg_mixed()
        if (outer > 0 && prev_it > 0 && prev_good && c0->h_st->rr > 0.0 && c0->h_st->beta > 0.0)
            pcoef = c0->h_st->beta / (c0->h_st->rr * (scale / prev_scale));
        int it = 0;
        rc = D32::cg(d, 5, false, eps, max_iter - total, &it, nullptr, pcoef);
        if (rc != LGT_OK && rc != LGT_ENOCONV) return rc;
        prev_scale = scale;
        prev_it = it;
        total += it;
        outer++;
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t off = D64::spinor_off(c), cnt = D64::spinor_n(c);
            LAUNCH(c, LGT_K_CG_BLAS, up_axpy_kernel, stream_blocks(c, cnt), 256, cnt, (double2*)c->ws[0] + off, (const float2*)c->ws32[1] + off, 1.0 / scale);
        }
        if ((rc = D64::dslash(d, 0, 3, 0)) != LGT_OK) return rc;  // t = D x
        if ((rc = D64::dslash(d, 3, 2, 1)) != LGT_OK) return rc;  // q = D^dag t
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t off = D64::spinor_off(c), cnt = D64::spinor_n(c);
            LAUNCH(c, LGT_K_CG_BLAS, residual_kernel, stream_blocks(c, cnt), 256, cnt, (const double2*)D64::fld(c, ib) + off,
                   (const double2*)c->ws[2] + off, (double2*)c->ws[1] + off, c->scal + 3, c->partials, c->counter, D64::zmask(c));
        }
        const double rr_before = rr;
        if ((rc = read_sum(rr)) != LGT_OK) return rc;
        prev_good = rr <= 100.0 * eps * eps * rr_before;
    }
    (void)want_y;  // Y = D x is what the last residual evaluation left in ws[3]
    if (iters) *iters = total;
    if (conv != LGT_OK) return dd_fail(d, LGT_ENOCONV, "mixed-precision CG did not reach the tolerance");
    return LGT_OK;
}

// (M^dag M) x_e = phi_e on the slabs in mixed precision: eo_cg_mixed()'s defect correction with the decomposed fp32 CG
// inside and the all-reduced true fp64 residual outside.  fp64 half fields: b = even of (4,5), x = even of (0,1),
// r = odd of (4,5), q = field 6, u = even of (2,3), t = field 7 (the assignment of DdOps<double>::eo_solve).
int dd_eo_cg_mixed(lgt_dd* d, double tol, int max_iter, int* iters) {
    typedef DdOps<double> D64;
    typedef DdOps<float> D32;
    int rc;
    const int n = (int)d->rk.size();
    std::vector<double*> slot;
    for (int i = 0; i < n; i++) {
        lgt_ctx* c = d->rk[i];
        const size_t nh = (size_t)12 * c->g.Vhs, nu = (size_t)2 * 36 * c->g.Vhs;
        if (!c->Ucb32) {
            DD_CU(cudaMalloc(&c->Ucb32, nu * sizeof(float2)));
            DD_CU(cudaMalloc(&c->eo32, 6 * nh * sizeof(float2)));
            DD_CU(cudaMemsetAsync(c->eo32, 0, 6 * nh * sizeof(float2), d->stream));
            c->ucb32_valid = false;
        }
        if (!c->ucb32_valid) {
            LAUNCH(c, LGT_K_OTHER, down_convert_kernel, stream_blocks(c, nu), 256, nu, (const double2*)c->Ucb, (float2*)c->Ucb32, 1.0);
            c->ucb32_valid = true;
        }
        const size_t off = D64::half_off(c), cnt = D64::half_n(c);
        DD_CU(cudaMemsetAsync(D64::hXe(c), 0, nh * sizeof(double2), d->stream));
        DD_CU(cudaMemcpyAsync(D64::hR(c), D64::hB(c), nh * sizeof(double2), cudaMemcpyDeviceToDevice, d->stream));
        LAUNCH(c, LGT_K_OTHER, (redot_kernel<double>), stream_blocks(c, cnt), 256, cnt, (const double2*)D64::hB(c) + off,
               (const double2*)D64::hB(c) + off, c->scal + 3, c->partials, c->counter, D64::zmask_half(c));
        slot.push_back(c->scal + 3);
    }
    lgt_ctx* c0 = d->rk[0];
    auto read_sum = [&](double& out) -> int {
        int r2 = dd_allreduce(d, slot.data(), 1);
        if (r2 != LGT_OK) return r2;
        DD_CU(cudaMemcpyAsync(c0->h_scal + 3, c0->scal + 3, sizeof(double), cudaMemcpyDeviceToHost, d->stream));
        DD_CU(cudaStreamSynchronize(d->stream));
        out = c0->h_scal[3];
        return LGT_OK;
    };
    double bb = 0.0;
    if ((rc = read_sum(bb)) != LGT_OK) return rc;
    double rr = bb;
    int total = 0, outer = 0, conv = LGT_OK, prev_it = 0;
    double prev_scale = 1.0;
    bool prev_good = false;
    while (bb > 0.0 && rr > tol * tol * bb) {
        if (total >= max_iter || outer >= 40) {
            conv = LGT_ENOCONV;
            break;
        }
        const double scale = 1.0 / sqrt(rr);
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t nh = (size_t)12 * c->g.Vhs;
            LAUNCH(c, LGT_K_CG_BLAS, down_convert_kernel, stream_blocks(c, nh), 256, nh, (const double2*)D64::hR(c), D32::template F<0>(c), scale);
        }
        double eps = 0.25 * tol * sqrt(bb / rr);
        if (eps < c0->inner_tol) eps = c0->inner_tol;
        double pcoef = 0.0;  // reliable update instead of a restart, as in eo_cg_mixed()
        if (outer > 0 && prev_it > 0 && prev_good && c0->h_st->rr > 0.0 && c0->h_st->beta > 0.0)
            pcoef = c0->h_st->beta / (c0->h_st->rr * (scale / prev_scale));
        CgState st32;
        rc = D32::eo_cg_loop(d, D32::template F<0>, D32::template F<1>, D32::template F<2>, D32::template F<3>, D32::template F<4>,
                             D32::template F<5>, eps, max_iter - total, &st32, pcoef);
        if (rc != LGT_OK) return rc;
        prev_scale = scale;
        prev_it = st32.iter;
        total += st32.iter;
        outer++;
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t off = D64::half_off(c), cnt = D64::half_n(c);
            LAUNCH(c, LGT_K_CG_BLAS, up_axpy_kernel, stream_blocks(c, cnt), 256, cnt, (double2*)D64::hXe(c) + off,
                   (const float2*)D32::template F<1>(c) + off, 1.0 / scale);
        }
        if ((rc = D64::hop_all(d, false, D64::hXe, nullptr, D64::hT, 0, 0, false)) != LGT_OK) return rc;  // u = M x
        if ((rc = D64::hop_all(d, true, D64::hT, D64::hXe, D64::hYe, 0, 0, true)) != LGT_OK) return rc;
        if ((rc = D64::hop_all(d, false, D64::hYe, nullptr, D64::hT, 1, 0, false)) != LGT_OK) return rc;  // q = M^dag u
        if ((rc = D64::hop_all(d, true, D64::hT, D64::hYe, D64::hP, 1, 0, true)) != LGT_OK) return rc;
        for (int i = 0; i < n; i++) {
            lgt_ctx* c = d->rk[i];
            const size_t off = D64::half_off(c), cnt = D64::half_n(c);
            LAUNCH(c, LGT_K_CG_BLAS, residual_kernel, stream_blocks(c, cnt), 256, cnt, (const double2*)D64::hB(c) + off,
                   (const double2*)D64::hP(c) + off, (double2*)D64::hR(c) + off, c->scal + 3, c->partials, c->counter, D64::zmask_half(c));
        }
        const double rr_old = rr;
        if ((rc = read_sum(rr)) != LGT_OK) return rc;
        for (int i = 0; i < n; i++) mixed_inner_fallback(d->rk[i], rr_old, rr, eps);  // the same decision on every rank: rr is the global sum
        prev_good = rr <= 100.0 * eps * eps * rr_old;
    }
    if (iters) *iters = total;
    if (conv != LGT_OK) return dd_fail(d, LGT_ENOCONV, "mixed-precision even/odd CG did not reach the tolerance");
    return LGT_OK;
}

int dd_solve(lgt_dd* d, int ib, bool want_y, double tol, int max_iter, int* iters) {
    if (d->prec == LGT_F64 && d->rk[0]->solver == LGT_SOLVER_MIXED_CG) return dd_cg_mixed(d, ib, want_y, tol, max_iter, iters);
    return DD_DISPATCH(d, cg, d, ib, want_y, tol, max_iter, iters, nullptr);
}

}  // namespace

#define CHECK_DD(d)               \
    if (!(d)) return LGT_EINVAL;  \
    DeviceGuard guard_((d)->device)

extern "C" {

const char* lgt_dd_last_error(const lgt_dd* d) { return d ? d->err.c_str() : g_dd_create_error.c_str(); }

int lgt_dd_destroy(lgt_dd* d) {
    if (!d) return LGT_OK;
    DeviceGuard guard(d->device);
    cudaStreamSynchronize(d->stream);
    if (d->comm && g_nccl.CommDestroy) g_nccl.CommDestroy(d->comm);
    for (int f = 0; f < 2; f++)
        for (int sd = 0; sd < 2; sd++)
            if (d->ipc_open[f][sd]) cudaIpcCloseMemHandle(d->ipc_peer[f][sd]);
    if (d->h_stage) cudaFreeHost(d->h_stage);
    if (d->h_sum) cudaFreeHost(d->h_sum);
    if (d->d_stage) cudaFree(d->d_stage);
    for (lgt_ctx* c : d->rk) lgt_destroy(c);
    delete d;
    return LGT_OK;
}

int lgt_dd_halo_plan(int nranks, int rank, int lt_local, int plan[8]) {
    if (!plan || nranks < 1 || rank < 0 || rank >= nranks || lt_local < 1) return LGT_EINVAL;
    const HaloPlan p = halo_plan(nranks, rank, lt_local);
    for (int k = 0; k < 2; k++) {
        plan[k] = p.send_peer[k];
        plan[2 + k] = p.send_slice[k];
        plan[4 + k] = p.recv_peer[k];
        plan[6 + k] = p.recv_slice[k];
    }
    return LGT_OK;
}

int lgt_dd_set_host_transport(lgt_dd* d, lgt_dd_sendrecv_fn sendrecv, lgt_dd_allreduce_fn allreduce, void* user) {
    CHECK_DD(d);
    if (!sendrecv || !allreduce) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_host_transport: null callback");
    if (d->rk.size() != 1) return dd_fail(d, LGT_ESTATE, "lgt_dd_set_host_transport: the host transport serves one rank per process");
    if (d->comm) return dd_fail(d, LGT_ESTATE, "lgt_dd_set_host_transport: this group already uses NCCL");
    d->host_sendrecv = sendrecv;
    d->host_allreduce = allreduce;
    d->host_user = user;
    d->links_ghost_valid = false;
    return LGT_OK;
}

int lgt_dd_create(lgt_dd** out, const int dims[4], int nranks, int nlocal, const int* local_ranks, double beta, double kappa,
                  const int bc[4], int precision, int device, void* cuda_stream) {
    lgt_dd* d = nullptr;
    if (!out || !dims || !bc || !local_ranks) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: null argument");
    *out = nullptr;
    if (nranks < 1 || nlocal < 1 || nlocal > nranks || nlocal > 8) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: need 1 <= nlocal <= min(nranks, 8)");
    if (nlocal != nranks && nlocal != 1) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: either every rank is local or exactly one is");
    for (int m = 0; m < 4; m++)
        if (dims[m] < 1) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: dims must be >= 1");
    if (dims[3] % nranks != 0) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: Lt must be a multiple of the number of ranks");
    const long long V3 = (long long)dims[0] * dims[1] * dims[2];
    if (V3 % 32 != 0) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: Lx*Ly*Lz must be a multiple of 32 (a time slice is then one contiguous run)");
    for (int i = 0; i < nlocal; i++) {
        if (local_ranks[i] < 0 || local_ranks[i] >= nranks) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: bad local rank number");
        for (int j = 0; j < i; j++)
            if (local_ranks[j] == local_ranks[i]) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create: duplicate local rank number");
    }
    d = new lgt_dd();
    d->nranks = nranks;
    d->Lt_loc = dims[3] / nranks;
    d->V3 = (int)V3;
    d->prec = precision;
    d->device = device;
    d->stream = (cudaStream_t)cuda_stream;
    const int ldims[4] = {dims[0], dims[1], dims[2], d->Lt_loc + 2};
    for (int i = 0; i < nlocal; i++) {
        lgt_ctx* c = nullptr;
        int rc = lgt_create(&c, ldims, beta, kappa, bc, precision, device, cuda_stream);
        if (rc != LGT_OK) {
            g_dd_create_error = std::string("lgt_dd_create: ") + lgt_last_error(nullptr);
            lgt_dd_destroy(d);
            return rc;
        }
        c->g.s_begin = d->V3;
        c->g.s_end = c->g.V - d->V3;
        c->g.t_off = local_ranks[i] * d->Lt_loc - 1;
        c->g.Lt_glob = dims[3];
        c->g.site_off = (local_ranks[i] * d->Lt_loc - 1) * d->V3;
        c->g.h_begin = d->V3 / 2;
        c->g.h_end = c->g.Vh - d->V3 / 2;
        c->g.swz_Z = 0;
        c->dd_links_valid = &d->links_ghost_valid;
        d->rk.push_back(c);
        d->rank_of.push_back(local_ranks[i]);
        // the unit field again, now with the boundary sign at the right global time slice
        rc = precision == LGT_F64 ? Ops<double>::unit_links(c) : Ops<float>::unit_links(c);
        if (rc != LGT_OK) {
            g_dd_create_error = "lgt_dd_create: " + c->err;
            lgt_dd_destroy(d);
            return rc;
        }
    }
    d->links_ghost_valid = true;  // the unit field fills the ghost slices too
    *out = d;
    return LGT_OK;
}

int lgt_dd_create_grid(lgt_dd** out, const int dims[4], const int grid[2], int nlocal, const int* local_ranks, double beta, double kappa,
                       const int bc[4], int precision, int device, void* cuda_stream) {
    lgt_dd* d = nullptr;
    if (!out || !dims || !grid || !bc || !local_ranks) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: null argument");
    *out = nullptr;
    const int Pt = grid[0], Pz = grid[1];
    if (Pt < 1 || Pz < 1) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: grid = {Pt, Pz} with both >= 1");
    const int nranks = Pt * Pz;
    if (nlocal < 1 || nlocal > nranks || nlocal > 8) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: need 1 <= nlocal <= min(Pt * Pz, 8)");
    if (nlocal != nranks && nlocal != 1) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: either every rank is local or exactly one is");
    for (int m = 0; m < 4; m++)
        if (dims[m] < 1) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: dims must be >= 1");
    if (dims[3] % Pt != 0 || dims[2] % Pz != 0) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: Lt must be a multiple of Pt and Lz of Pz");
    const long long xy = (long long)dims[0] * dims[1];
    if (xy % 32 != 0) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: Lx*Ly must be a multiple of 32 (an xy plane is then whole layout blocks)");
    for (int i = 0; i < nlocal; i++) {
        if (local_ranks[i] < 0 || local_ranks[i] >= nranks) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: bad local rank number");
        for (int j = 0; j < i; j++)
            if (local_ranks[j] == local_ranks[i]) return dd_fail(nullptr, LGT_EINVAL, "lgt_dd_create_grid: duplicate local rank number");
    }
    d = new lgt_dd();
    d->nranks = nranks;
    d->Pt = Pt;
    d->Pz = Pz;
    d->Lt_loc = dims[3] / Pt;
    d->Lz_loc = dims[2] / Pz;
    d->LxLy = (int)xy;
    d->V3 = (int)(xy * (d->Lz_loc + 2));  // a LOCAL time slice, ghost z planes included
    d->Vglob = xy * dims[2] * dims[3];
    d->prec = precision;
    d->device = device;
    d->stream = (cudaStream_t)cuda_stream;
    const int ldims[4] = {dims[0], dims[1], d->Lz_loc + 2, d->Lt_loc + 2};
    for (int i = 0; i < nlocal; i++) {
        lgt_ctx* c = nullptr;
        int rc = lgt_create(&c, ldims, beta, kappa, bc, precision, device, cuda_stream);
        if (rc != LGT_OK) {
            g_dd_create_error = std::string("lgt_dd_create_grid: ") + lgt_last_error(nullptr);
            lgt_dd_destroy(d);
            return rc;
        }
        const int pt = local_ranks[i] / Pz, pz = local_ranks[i] % Pz;
        c->g.s_begin = d->V3;
        c->g.s_end = c->g.V - d->V3;
        c->g.t_off = pt * d->Lt_loc - 1;
        c->g.Lt_glob = dims[3];
        c->g.z_lo = 1;
        c->g.z_hi = d->Lz_loc + 1;
        c->g.z_off = pz * d->Lz_loc - 1;
        c->g.Lz_glob = dims[2];
        c->g.site_off = 0;  // grid ranks number their elements through global_site()
        c->g.h_begin = d->V3 / 2;
        c->g.h_end = c->g.Vh - d->V3 / 2;
        c->g.swz_Z = 0;
        c->dd_links_valid = &d->links_ghost_valid;
        d->rk.push_back(c);
        d->rank_of.push_back(local_ranks[i]);
        rc = precision == LGT_F64 ? Ops<double>::unit_links(c) : Ops<float>::unit_links(c);
        if (rc != LGT_OK) {
            g_dd_create_error = "lgt_dd_create_grid: " + c->err;
            lgt_dd_destroy(d);
            return rc;
        }
    }
    d->links_ghost_valid = true;  // the unit field fills the ghost slices and planes too
    *out = d;
    return LGT_OK;
}

int lgt_dd_nccl_unique_id(void* id128) {
    if (!id128) return LGT_EINVAL;
    if (!g_nccl.load()) return dd_fail(nullptr, LGT_ECUDA, "lgt_dd_nccl_unique_id: libnccl.so.2 not found");
    NcclApi::UniqueId id;
    if (g_nccl.GetUniqueId(&id) != 0) return dd_fail(nullptr, LGT_ECUDA, "ncclGetUniqueId failed");
    memcpy(id128, &id, sizeof id);
    return LGT_OK;
}
int lgt_dd_nccl_init(lgt_dd* d, const void* id128) {
    CHECK_DD(d);
    if (!id128) return dd_fail(d, LGT_EINVAL, "lgt_dd_nccl_init: null id");
    if (d->rk.size() != 1) return dd_fail(d, LGT_ESTATE, "lgt_dd_nccl_init: the NCCL transport serves one rank per process");
    if (d->comm) return dd_fail(d, LGT_ESTATE, "lgt_dd_nccl_init: already initialised");
    if (d->host_sendrecv) return dd_fail(d, LGT_ESTATE, "lgt_dd_nccl_init: this group already uses a host transport");
    if (!g_nccl.load()) return dd_fail(d, LGT_ECUDA, "lgt_dd_nccl_init: libnccl.so.2 not found");
    NcclApi::UniqueId id;
    memcpy(&id, id128, sizeof id);
    DD_NCCL(g_nccl.CommInitRank(&d->comm, d->nranks, id, d->rank_of[0]));
    d->links_ghost_valid = false;
    return LGT_OK;
}

int lgt_dd_set_halo_mode(lgt_dd* d, int mode) {
    CHECK_DD(d);
    if (mode != LGT_DD_EXCHANGE && mode != LGT_DD_PUSH && mode != LGT_DD_OVERLAP && mode != LGT_DD_HALF)
        return dd_fail(d, LGT_EINVAL, "lgt_dd_set_halo_mode: unknown mode");
    if (mode == LGT_DD_PUSH && d->Pz > 0) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_halo_mode: LGT_DD_PUSH is for time slabs; a (Pt, Pz) grid exchanges");
    if (mode == LGT_DD_PUSH && d->rk.size() != (size_t)d->nranks && d->nranks > 1)
        for (int f = 0; f < 2; f++)
            for (int s = 0; s < 2; s++)
                if (!d->ipc_peer[f][s]) return dd_fail(d, LGT_ESTATE, "lgt_dd_set_halo_mode: LGT_DD_PUSH needs the neighbours' buffers (lgt_dd_ipc_import)");
    d->halo_mode = mode;
    return LGT_OK;
}
// 2 x 64 bytes: the CUDA IPC handles of this rank's r and t fields (ws[1], ws[3])
int lgt_dd_ipc_export(lgt_dd* d, void* handles128) {
    CHECK_DD(d);
    if (!handles128) return dd_fail(d, LGT_EINVAL, "lgt_dd_ipc_export: null pointer");
    if (d->rk.size() != 1) return dd_fail(d, LGT_ESTATE, "lgt_dd_ipc_export: one rank per process");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handle size");
    cudaIpcMemHandle_t h[2];
    DD_CU(cudaIpcGetMemHandle(&h[0], d->rk[0]->ws[1]));
    DD_CU(cudaIpcGetMemHandle(&h[1], d->rk[0]->ws[3]));
    memcpy(handles128, h, sizeof h);
    return LGT_OK;
}
int lgt_dd_ipc_import(lgt_dd* d, const void* lo_handles128, const void* hi_handles128) {
    CHECK_DD(d);
    if (!lo_handles128 || !hi_handles128) return dd_fail(d, LGT_EINVAL, "lgt_dd_ipc_import: null pointer");
    if (d->rk.size() != 1 || d->nranks < 2) return dd_fail(d, LGT_ESTATE, "lgt_dd_ipc_import: for one rank per process and at least two ranks");
    if (d->ipc_peer[0][0]) return dd_fail(d, LGT_ESTATE, "lgt_dd_ipc_import: already imported");
    cudaIpcMemHandle_t lo[2], hi[2];
    memcpy(lo, lo_handles128, sizeof lo);
    memcpy(hi, hi_handles128, sizeof hi);
    const bool same_peer = d->nranks == 2;  // both neighbours are the one other rank: map its buffers once
    for (int f = 0; f < 2; f++) {
        DD_CU(cudaIpcOpenMemHandle(&d->ipc_peer[f][0], lo[f], cudaIpcMemLazyEnablePeerAccess));
        d->ipc_open[f][0] = true;
        if (same_peer) {
            d->ipc_peer[f][1] = d->ipc_peer[f][0];
        } else {
            DD_CU(cudaIpcOpenMemHandle(&d->ipc_peer[f][1], hi[f], cudaIpcMemLazyEnablePeerAccess));
            d->ipc_open[f][1] = true;
        }
    }
    return LGT_OK;
}

int lgt_dd_local_ranks(const lgt_dd* d) { return d ? (int)d->rk.size() : 0; }
lgt_ctx* lgt_dd_rank(lgt_dd* d, int local_index) {
    if (!d || local_index < 0 || local_index >= (int)d->rk.size()) return nullptr;
    return d->rk[local_index];
}

int lgt_dd_dslash(lgt_dd* d, const void* const* in, void* const* out, int dagger) {
    CHECK_DD(d);
    if (!in || !out) return dd_fail(d, LGT_EINVAL, "lgt_dd_dslash: null pointer");
    for (size_t i = 0; i < d->rk.size(); i++) {
        if (!in[i] || !out[i] || in[i] == out[i]) return dd_fail(d, LGT_EINVAL, "lgt_dd_dslash: in and out must be distinct non-null buffers");
        DD_RK(i, DISPATCH(d->rk[i], to_native, d->rk[i], in[i], d->rk[i]->ws[4], 12));
    }
    int rc = DD_DISPATCH(d, dslash, d, 4, 5, dagger ? 1 : 0);
    if (rc != LGT_OK) return rc;
    for (size_t i = 0; i < d->rk.size(); i++) DD_RK(i, DISPATCH(d->rk[i], from_native, d->rk[i], d->rk[i]->ws[5], out[i], 12));
    return LGT_OK;
}
int lgt_dd_cg(lgt_dd* d, const void* const* b, void* const* x, double tol, int max_iter, int* iters, double* rel_resid) {
    CHECK_DD(d);
    if (!b || !x) return dd_fail(d, LGT_EINVAL, "lgt_dd_cg: null pointer");
    if (!(tol >= 0.0) || max_iter < 0) return dd_fail(d, LGT_EINVAL, "lgt_dd_cg: bad tol / max_iter");
    for (size_t i = 0; i < d->rk.size(); i++) {
        if (!b[i] || !x[i]) return dd_fail(d, LGT_EINVAL, "lgt_dd_cg: null pointer");
        DD_RK(i, DISPATCH(d->rk[i], to_native, d->rk[i], b[i], d->rk[i]->ws[5], 12));
    }
    int conv = DD_DISPATCH(d, cg, d, 5, false, tol, max_iter, iters, rel_resid);
    if (conv != LGT_OK && conv != LGT_ENOCONV) return conv;
    for (size_t i = 0; i < d->rk.size(); i++) DD_RK(i, DISPATCH(d->rk[i], from_native, d->rk[i], d->rk[i]->ws[0], x[i], 12));
    return conv;
}
int lgt_dd_action(lgt_dd* d, double tol, int max_iter, double* S_g, double* S_F, double* K, int* cg_iters) {
    CHECK_DD(d);
    return DD_DISPATCH(d, action, d, tol, max_iter, S_g, S_F, K, cg_iters);
}
int lgt_dd_md_kick(lgt_dd* d, double eps, double tol, int max_iter, int* cg_iters) {
    CHECK_DD(d);
    return DD_DISPATCH(d, kick, d, eps, tol, max_iter, cg_iters);
}
int lgt_dd_md_drift(lgt_dd* d, double eps) {
    CHECK_DD(d);
    return DD_DISPATCH(d, drift, d, eps);
}
int lgt_dd_md_trajectory(lgt_dd* d, int nsteps, double dt, double tol, int max_iter, double* H_initial, double* H_final, long* cg_iters) {
    CHECK_DD(d);
    if (nsteps < 0) return dd_fail(d, LGT_EINVAL, "lgt_dd_md_trajectory: nsteps < 0");
    int rc, it = 0, conv = LGT_OK;
    long total = 0;
    double sg, sf, k;
#define DD_STEP(call)                      \
    do {                                   \
        it = 0;                            \
        rc = (call);                       \
        if (rc == LGT_ENOCONV) conv = rc;  \
        else if (rc != LGT_OK) return rc;  \
    } while (0)
    if (H_initial) {
        DD_STEP(DD_DISPATCH(d, action, d, tol, max_iter, &sg, &sf, &k, &it));
        *H_initial = k + sg + sf;
    }
    rc = DD_DISPATCH(d, integrate, d, nsteps, dt, tol, max_iter, &total);
    if (rc == LGT_ENOCONV) conv = rc;
    else if (rc != LGT_OK) return rc;
    if (H_final) {
        DD_STEP(DD_DISPATCH(d, action, d, tol, max_iter, &sg, &sf, &k, &it));
        *H_final = k + sg + sf;
    }
#undef DD_STEP
    if (cg_iters) *cg_iters = total;
    DD_CU(cudaStreamSynchronize(d->stream));
    return conv;
}

int lgt_dd_set_fermion_action(lgt_dd* d, int action) {
    CHECK_DD(d);
    if (action != LGT_ACTION_FULL && action != LGT_ACTION_EO) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_fermion_action: unknown action");
    if (action == LGT_ACTION_EO) {
        const Geom& g = d->rk[0]->g;
        if (g.L[0] % 2 || g.L[1] % 2 || g.L[2] % 2 || d->Lt_loc % 2 || d->V3 % 64)
            return dd_fail(d, LGT_EINVAL, "lgt_dd_set_fermion_action: the even/odd action needs even extents, an even number of time slices "
                                          "per slab and Lx*Ly*Lz a multiple of 64");
        if (d->Pz > 0 && d->LxLy % 64)  // (Lz_loc + 2 even is the g.L[2] check above)
            return dd_fail(d, LGT_EINVAL, "lgt_dd_set_fermion_action: on a (Pt, Pz) grid the even/odd action needs Lx*Ly a multiple of 64 "
                                          "(the z faces of a half field are then whole layout blocks)");
    }
    for (lgt_ctx* c : d->rk) c->action = action;
    return LGT_OK;
}
int lgt_dd_set_integrator(lgt_dd* d, int integrator, int n_inner) {
    CHECK_DD(d);
    if (integrator != LGT_INT_LEAPFROG && integrator != LGT_INT_OMELYAN && integrator != LGT_INT_SEXTON_WEINGARTEN)
        return dd_fail(d, LGT_EINVAL, "lgt_dd_set_integrator: unknown integrator");
    if (integrator == LGT_INT_SEXTON_WEINGARTEN && n_inner < 1) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_integrator: n_inner must be >= 1");
    for (lgt_ctx* c : d->rk) {
        c->integrator = integrator;
        c->n_inner = integrator == LGT_INT_SEXTON_WEINGARTEN ? n_inner : 1;
    }
    return LGT_OK;
}
int lgt_dd_set_smearing(lgt_dd* d, int n_levels, double rho) {
    CHECK_DD(d);
    if (n_levels < 0 || n_levels > LGT_MAX_SMEAR) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_smearing: n_levels must be in 0..8");
    if (n_levels > 0 && !(rho >= 0.0)) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_smearing: rho must be >= 0");
    for (lgt_ctx* c : d->rk) {
        c->nsmear = n_levels;
        c->rho = n_levels ? rho : 0.0;
        c->usm_valid = c->u32_valid = c->ucb_valid = c->ucb32_valid = false;
    }
    return LGT_OK;
}
int lgt_dd_set_solver(lgt_dd* d, int solver, double inner_tol) {
    CHECK_DD(d);
    if (solver != LGT_SOLVER_CG && solver != LGT_SOLVER_MIXED_CG) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_solver: unknown solver");
    if (solver == LGT_SOLVER_MIXED_CG && d->prec != LGT_F64) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_solver: mixed precision needs an LGT_F64 group");
    if (solver == LGT_SOLVER_MIXED_CG && !(inner_tol > 0.0 && inner_tol < 1.0)) return dd_fail(d, LGT_EINVAL, "lgt_dd_set_solver: inner_tol must be in (0, 1)");
    for (lgt_ctx* c : d->rk) {
        c->solver = solver;
        if (solver == LGT_SOLVER_MIXED_CG) c->inner_tol = inner_tol;
    }
    return LGT_OK;
}

int lgt_dd_hmc_trajectory(lgt_dd* d, int nsteps, double dt, double tol, int max_iter, unsigned long long seed, unsigned trajectory,
                          double* dH, int* accepted, long* cg_iters, double* H_initial) {
    CHECK_DD(d);
    if (nsteps < 0) return dd_fail(d, LGT_EINVAL, "lgt_dd_hmc_trajectory: nsteps < 0");
    return DD_DISPATCH(d, hmc_trajectory, d, nsteps, dt, tol, max_iter, seed, trajectory, dH, accepted, cg_iters, H_initial);
}

}  // extern "C"
