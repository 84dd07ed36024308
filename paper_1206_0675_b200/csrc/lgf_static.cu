// lgf_static.cu -- lgf_measure_static: F and theta (eqs. 3, 5-7) of a configuration in the canonical
// layout WITHOUT any allocation: no context, no cudaMalloc / cudaFree / allocating library call.  For callers that
// cannot allocate -- code under CUDA-graph capture, tight serving loops, harnesses that forbid it.
//
// It is the a1 kernel (k_delta, lgf_links.cu) reading the caller's canonical array directly, with the per-block
// partial sums -- the scratch memory every reduction of this library needs -- in a file-scope device array of a
// fixed, modest size instead of a context's buffer:
//     LGF_STATIC_MAX_SITES = 2^21 sites (32^4 and 32^3 x 64 fit), 256 sites per block -> 8192 blocks x 2 doubles = 128 KB,
// held by every GPU that loads liblgf.so until the process exits.  Larger lattices are refused (LGF_EINVAL): use a
// context (lgf_create / lgf_measure).
//
// The array is SHARED by all calls and keeps the last call's contents.  Nothing in it has to start at zero: a
// call writes entries 0 .. nb-1 and its final sum reads exactly those, so a stale tail from a larger lattice is
// never read.  Calls that overlap on the GPU (two streams, two host threads) race on it -- serialise them.
//
// In host code the array's name is a host-side stand-in, not a device address; the address the kernels get is
// taken with cudaGetSymbolAddress, once per device, with that device current (static_scratch()).
// Part of liblgf (CUDA path).  Shares nothing with oracle/.
#include <mutex>
#include <string>

#include "../../include/lgf.h"
#include "lgf_su3.cuh"

namespace lgf {

constexpr int STATIC_THREADS = 256;
constexpr long long STATIC_MAX_SITES = LGF_STATIC_MAX_SITES;
constexpr int STATIC_MAX_BLOCKS = (int)(STATIC_MAX_SITES / STATIC_THREADS);

static __device__ __align__(256) double g_static_scratch[2 * STATIC_MAX_BLOCKS];

// canonical layout: canon[((s*4 + mu)*9 + e)*2 + re/im]   (include/lgf.h)
template <class R>
__device__ __forceinline__ void load_link_canon(const C<R> *__restrict__ canon, long long s, int mu, C<R> (&u)[9]) {
    const C<R> *p = canon + (s * 4 + mu) * 9;
#pragma unroll
    for (int e = 0; e < 9; e++) u[e] = p[e];
}

// a1 on the canonical array: per-site Re tr U and tr(Delta Delta^dag), block sums into `scratch`
template <class R>
__global__ void __launch_bounds__(STATIC_THREADS) k_delta_canon(const C<R> *__restrict__ canon, Geom g, double *__restrict__ scratch) {
    __shared__ double sh[STATIC_THREADS / 32][2];
    const long long s = (long long)blockIdx.x * STATIC_THREADS + threadIdx.x;
    double f = 0.0, t = 0.0;
    if (s < g.V) {
        int c[4];
        site_coords(g, s, c);
        Herm<R> d = herm_zero<R>();
        R retr = 0;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            C<R> u[9];
            load_link_canon(canon, s, mu, u);
            retr += u[0].x + u[4].x + u[8].x;                       // eq. 3: Re tr U_mu(x)
            herm_sub(d, algebra_part(u));                           // - A_mu(x)
            load_link_canon(canon, site_bwd(g, s, c, mu), mu, u);
            herm_add(d, algebra_part(u));                           // + A_mu(x - mu)      (eq. 5)
        }
        f = (double)retr;
        t = (double)herm_norm2(d);                                  // eq. 6: tr(Delta Delta^dag)
    }
    block_sum2(f, t, sh);
    if (threadIdx.x == 0) {
        scratch[2 * blockIdx.x] = f;
        scratch[2 * blockIdx.x + 1] = t;
    }
}

// fixed-order sum of entries 0 .. nb-1 (bit-reproducible), eq. 3 / eq. 6 normalisation; out = (F, theta)
__global__ void __launch_bounds__(1024) k_static_finalize(const double *__restrict__ scratch, int nb, long long V,
                                                           double *__restrict__ out) {
    __shared__ double sh[32][2];
    double f = 0.0, t = 0.0;
    for (int i = threadIdx.x; i < nb; i += 1024) {
        f += scratch[2 * i];
        t += scratch[2 * i + 1];
    }
    block_sum2(f, t, sh);
    if (threadIdx.x == 0) {
        out[0] = f / (12.0 * (double)V);
        out[1] = t / (3.0 * (double)V);
    }
}

// device address of the scratch array on the CURRENT device, looked up once per device
static cudaError_t static_scratch(double **out) {
    constexpr int MAXDEV = 64;
    static std::mutex mu;
    static double *addr[MAXDEV] = {nullptr};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAXDEV) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        addr[dev] = p;
    }
    *out = addr[dev];
    return cudaSuccess;
}

}  // namespace lgf

using namespace lgf;

static thread_local std::string g_static_err;
static int static_fail(int code, const std::string &msg) {
    g_static_err = msg;
    return code;
}

extern "C" {

const char *lgf_static_last_error(void) { return g_static_err.c_str(); }

int lgf_measure_static(const int dims[4], int precision, const void *d_links, double *d_F_theta, void *cuda_stream) {
    if (!dims || !d_links || !d_F_theta) return static_fail(LGF_EINVAL, "lgf_measure_static: null argument");
    if (precision != LGF_FP32 && precision != LGF_FP64) return static_fail(LGF_EINVAL, "lgf_measure_static: bad precision");
    Geom g;
    long long S = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (dims[mu] < 1) return static_fail(LGF_EINVAL, "lgf_measure_static: bad lattice extent");
        g.L[mu] = dims[mu];
        g.S[mu] = S;
        S *= dims[mu];
        if (S > STATIC_MAX_SITES)
            return static_fail(LGF_EINVAL, "lgf_measure_static: lattice beyond LGF_STATIC_MAX_SITES = " + std::to_string(STATIC_MAX_SITES) +
                                               " sites (the fixed scratch array); use lgf_create / lgf_measure");
    }
    g.V = S;
    double *scratch = nullptr;
    cudaError_t e = static_scratch(&scratch);
    if (e != cudaSuccess) return static_fail(LGF_ECUDA, std::string("lgf_measure_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int nb = (int)((g.V + STATIC_THREADS - 1) / STATIC_THREADS);
    if (precision == LGF_FP64) k_delta_canon<double><<<nb, STATIC_THREADS, 0, stream>>>((const C<double> *)d_links, g, scratch);
    else k_delta_canon<float><<<nb, STATIC_THREADS, 0, stream>>>((const C<float> *)d_links, g, scratch);
    k_static_finalize<<<1, 1024, 0, stream>>>(scratch, nb, g.V, d_F_theta);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(LGF_ECUDA, std::string("lgf_measure_static: launch: ") + cudaGetErrorString(e));
    return LGF_OK;
}

}  // extern "C"
