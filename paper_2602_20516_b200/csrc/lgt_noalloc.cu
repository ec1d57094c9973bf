// lgt_plaquette_action_noalloc: the plaquette action (BASELINE.json configs[0]:
//   S_g = beta sum_x sum_{mu<nu} (1 - Re tr U_P(x) / 3),  U_P = U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x))
// for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// It is plaquette_kernel (kernels.cuh) with two changes: the links are read in the CANONICAL layout [V][4][3][3] the caller
// holds (no handle, no native copy), and the scratch of the deterministic reduction -- one double per block of 128 sites and
// the ticket counter -- lives in a file-scope __device__ array of fixed size instead of the handle's cudaMalloc'ed buffers.
// The array is part of the library image: every GPU that loads liblgt.so holds its 1 MiB + 256 B until the process exits.
//
// This file is a translation unit of its own and shares no state with lgt_api.cu; the existing entry points are unchanged.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "lgt.h"

namespace {

constexpr int NOALLOC_BLOCK = 128;                                                      // sites per block
constexpr int NOALLOC_MAX_BLOCKS = LGT_NOALLOC_MAX_SITES / NOALLOC_BLOCK;               // 131072 block partials
constexpr int NOALLOC_COUNTER_AT = NOALLOC_MAX_BLOCKS;                                  // ticket counter behind the partials
constexpr int NOALLOC_SCRATCH_DOUBLES = NOALLOC_MAX_BLOCKS + 32;                        // + one 256-byte line for the counter

// In HOST code this name is a host-side stand-in, not a device address: noalloc_scratch_on() below resolves it once per
// device with cudaGetSymbolAddress and the kernel is given that pointer.
static __device__ __align__(256) double noalloc_scratch[NOALLOC_SCRATCH_DOUBLES];

struct NoallocGeom {
    int L[4];
    int V;
};

template <class T> struct C2;
template <> struct C2<double> { typedef double2 type; };
template <> struct C2<float> { typedef float2 type; };

// c = a b (3 x 3 complex, row-major)
template <class T> __device__ __forceinline__ void mul33(const typename C2<T>::type* a, const typename C2<T>::type* b, typename C2<T>::type* c) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            T re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const typename C2<T>::type x = a[3 * i + k], y = b[3 * k + j];
                re = fma(x.x, y.x, re);
                re = fma(-x.y, y.y, re);
                im = fma(x.x, y.y, im);
                im = fma(x.y, y.x, im);
            }
            c[3 * i + j].x = re;
            c[3 * i + j].y = im;
        }
}

template <class T> __device__ __forceinline__ void load33(const typename C2<T>::type* U, int s, int mu, typename C2<T>::type* m) {
    const typename C2<T>::type* p = U + ((size_t)s * 4 + mu) * 9;
#pragma unroll
    for (int k = 0; k < 9; k++) m[k] = __ldg(p + k);
}

__device__ __forceinline__ int fwd_site(const NoallocGeom& g, const int x[4], int s, int mu) {
    int stride = 1;
    for (int k = 0; k < mu; k++) stride *= g.L[k];
    return (x[mu] == g.L[mu] - 1) ? s - (g.L[mu] - 1) * stride : s + stride;
}

// out[0] = S_g, out[1] = average plaquette (1 / 6V) sum Re tr U_P / 3.  Block sums by a fixed shuffle tree, block partials to
// scratch[blockIdx.x]; the block that draws the last ticket adds the partials in a fixed order: bitwise reproducible.
template <class T>
__global__ void __launch_bounds__(NOALLOC_BLOCK) plaquette_noalloc_kernel(NoallocGeom g, const typename C2<T>::type* __restrict__ U, double beta,
                                                                          double* __restrict__ out, double* scratch) {
    typedef typename C2<T>::type T2;
    __shared__ double warp_sums[NOALLOC_BLOCK / 32];
    __shared__ bool is_last;
    unsigned* counter = reinterpret_cast<unsigned*>(scratch + NOALLOC_COUNTER_AT);
    const int s = blockIdx.x * NOALLOC_BLOCK + threadIdx.x;
    double acc = 0.0;
    if (s < g.V) {
        int x[4], r = s;
#pragma unroll
        for (int k = 0; k < 4; k++) {
            x[k] = r % g.L[k];
            r /= g.L[k];
        }
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int smu = fwd_site(g, x, s, mu);
#pragma unroll
            for (int nu = mu + 1; nu < 4; nu++) {
                const int snu = fwd_site(g, x, s, nu);
                T2 a[9], b[9], t1[9], t2[9];
                load33<T>(U, s, mu, a);
                load33<T>(U, smu, nu, b);
                mul33<T>(a, b, t1);  // U_mu(x) U_nu(x+mu)
                load33<T>(U, s, nu, a);
                load33<T>(U, snu, mu, b);
                mul33<T>(a, b, t2);  // U_nu(x) U_mu(x+nu)
                T tr = 0;            // Re tr(t1 t2^dag)
#pragma unroll
                for (int k = 0; k < 9; k++) tr += t1[k].x * t2[k].x + t1[k].y * t2[k].y;
                acc += (double)tr;
            }
        }
        acc *= (1.0 / 3.0);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if (lane == 0) warp_sums[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double w = 0.0;
#pragma unroll
        for (int k = 0; k < NOALLOC_BLOCK / 32; k++) w += warp_sums[k];
        scratch[blockIdx.x] = w;
        __threadfence();
        is_last = (atomicAdd(counter, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // the last block: thread j sums partials j, j + 128, ... in order, then the same fixed tree over the 128 threads
    double t = 0.0;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += NOALLOC_BLOCK) t += __ldcg(scratch + i);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    __syncthreads();
    if (lane == 0) warp_sums[warp] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double sum = 0.0;
#pragma unroll
        for (int k = 0; k < NOALLOC_BLOCK / 32; k++) sum += warp_sums[k];
        out[0] = beta * (6.0 * (double)g.V - sum);
        out[1] = sum / (6.0 * (double)g.V);
        *counter = 0u;  // left clean for the next call (which clears it again anyway)
    }
}

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_setup_lock;
double* g_scratch_on[NOALLOC_MAX_DEVICES] = {};  // device address of noalloc_scratch, per device
thread_local char g_error[256] = "";

int noalloc_fail(int code, const char* what, const char* detail = nullptr) {
    if (detail) snprintf(g_error, sizeof g_error, "%s: %s", what, detail);
    else snprintf(g_error, sizeof g_error, "%s", what);
    return code;
}

// Set-up, once per device, with that device current: the device address of the file-scope array.
int noalloc_scratch_on(int device, double** ptr) {
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_on[device]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return noalloc_fail(LGT_ECUDA, "lgt_plaquette_action_noalloc: cudaGetSymbolAddress(noalloc_scratch) failed",
                                e != cudaSuccess ? cudaGetErrorString(e) : "null address");
        }
        g_scratch_on[device] = p;
    }
    *ptr = g_scratch_on[device];
    return LGT_OK;
}

}  // namespace

extern "C" {

const char* lgt_noalloc_last_error(void) { return g_error; }

int lgt_plaquette_action_noalloc(const int dims[4], double beta, int precision, int device, const void* U, double* out, void* cuda_stream) {
    if (!dims || !U || !out) return noalloc_fail(LGT_EINVAL, "lgt_plaquette_action_noalloc: null pointer");
    if (precision != LGT_F64 && precision != LGT_F32) return noalloc_fail(LGT_EINVAL, "lgt_plaquette_action_noalloc: precision must be LGT_F64 or LGT_F32");
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return noalloc_fail(LGT_EINVAL, "lgt_plaquette_action_noalloc: device out of range");
    long long V = 1;
    for (int k = 0; k < 4; k++) {
        if (dims[k] < 1) return noalloc_fail(LGT_EINVAL, "lgt_plaquette_action_noalloc: every extent must be at least 1");
        V *= dims[k];
        if (V > (long long)LGT_NOALLOC_MAX_SITES) {
            char msg[160];
            snprintf(msg, sizeof msg, "the lattice has more than LGT_NOALLOC_MAX_SITES = %d sites (the fixed scratch holds one partial per 128 sites)",
                     LGT_NOALLOC_MAX_SITES);
            return noalloc_fail(LGT_EINVAL, "lgt_plaquette_action_noalloc", msg);
        }
    }
    int before = -1;
    if (cudaGetDevice(&before) != cudaSuccess) return noalloc_fail(LGT_ECUDA, "lgt_plaquette_action_noalloc: cudaGetDevice failed");
    if (before != device && cudaSetDevice(device) != cudaSuccess) {
        cudaGetLastError();
        return noalloc_fail(LGT_ECUDA, "lgt_plaquette_action_noalloc: cudaSetDevice failed");
    }
    double* scratch = nullptr;
    int rc = noalloc_scratch_on(device, &scratch);
    if (rc == LGT_OK) {
        cudaStream_t stream = (cudaStream_t)cuda_stream;
        NoallocGeom g;
        for (int k = 0; k < 4; k++) g.L[k] = dims[k];
        g.V = (int)V;
        const int blocks = (int)((V + NOALLOC_BLOCK - 1) / NOALLOC_BLOCK);
        // the array keeps the last call's contents: the ticket counter must start at zero (an aborted launch may have left it
        // anywhere); the partials need no clearing, every block of this launch overwrites its own before the last block reads
        cudaError_t e = cudaMemsetAsync(scratch + NOALLOC_COUNTER_AT, 0, 256, stream);
        if (e == cudaSuccess) {
            if (precision == LGT_F64) plaquette_noalloc_kernel<double><<<blocks, NOALLOC_BLOCK, 0, stream>>>(g, (const double2*)U, beta, out, scratch);
            else plaquette_noalloc_kernel<float><<<blocks, NOALLOC_BLOCK, 0, stream>>>(g, (const float2*)U, beta, out, scratch);
            e = cudaGetLastError();
        }
        if (e != cudaSuccess) rc = noalloc_fail(LGT_ECUDA, "lgt_plaquette_action_noalloc: launch failed", cudaGetErrorString(e));
    }
    if (before != device) cudaSetDevice(before);
    return rc;
}

}  // extern "C"
