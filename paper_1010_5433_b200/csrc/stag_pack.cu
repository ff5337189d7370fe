// stag_pack.cu — a1: canonical fp64 links -> packed hopping matrices; vector format
// conversion.  Setup work, done once per gauge field, so written for clarity:
// canonical (AoS) reads are strided, packed writes are coalesced.
//   PAPER.md:109  12-real storage: "only the first two rows are stored"
//   PAPER.md:113  b = (float)a   (fp32 copies are a round-to-nearest cast of the fp64 input)
//   PAPER.md:119  "blocks of threads ... use contiguous regions of device memory" -> planes
#include <type_traits>

#include "stag_dslash.cuh"

namespace stag {

template <typename T> struct Chunk;
template <> struct Chunk<double> { typedef double2 type; static constexpr int reals = 2; };
template <> struct Chunk<float> { typedef float4 type; static constexpr int reals = 4; };

// write `n` reals m[0..n) of site e as 16-byte chunk planes (+ 8-byte tail for fp32, n%4==2)
template <int N>
__device__ __forceinline__ void write_planes(char *base, int Vh, int e, const double (&m)[18],
                                             double /*tag*/) {
    double2 *p = reinterpret_cast<double2 *>(base) + e;
#pragma unroll
    for (int k = 0; k < N / 2; ++k) p[(size_t)k * Vh] = make_double2(m[2 * k], m[2 * k + 1]);
}
template <int N>
__device__ __forceinline__ void write_planes(char *base, int Vh, int e, const double (&m)[18],
                                             float /*tag*/) {
    float4 *p = reinterpret_cast<float4 *>(base) + e;
#pragma unroll
    for (int k = 0; k < N / 4; ++k)
        p[(size_t)k * Vh] = make_float4((float)m[4 * k], (float)m[4 * k + 1],
                                        (float)m[4 * k + 2], (float)m[4 * k + 3]);
    if (N % 4 == 2)
        reinterpret_cast<float2 *>(base + (size_t)Vh * 16 * (N / 4))[e] =
            make_float2((float)m[N - 2], (float)m[N - 1]);
}

// N3 split-double: b = (float)a, c = (float)(a - (double)b), each in the fp32 planes
// layout; `base` = this (parity, direction)'s b planes, base + c_off = its c planes.
struct SplitTag {};
template <int N>
__device__ __forceinline__ void write_planes_split(char *base, size_t c_off, int Vh, int e, const double (&m)[18]) {
    double lo[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) lo[k] = m[k] - (double)(float)m[k];
    write_planes<N>(base, Vh, e, m, 0.0f);
    write_planes<N>(base + c_off, Vh, e, lo, 0.0f);
}

// blockIdx.y = p*8 + d.  T = double | float | SplitTag.
template <typename T, int RECON>
__global__ void __launch_bounds__(128)
gauge_pack_kernel(const Geom g, const double *__restrict__ canon, char *__restrict__ packed,
                  int *__restrict__ not_su3) {
    const int e = blockIdx.x * 128 + threadIdx.x;
    if (e >= g.Vh) return;
    const int par = blockIdx.y >> 3, d = blockIdx.y & 7, mu = d >> 1, bwd = d & 1;
    const Site s = site_of(g, e, par);
    const int x[4] = {s.x0, s.x1, s.x2, s.x3};
    int stride = 1, phase_sum = 0;
    for (int nu = 0; nu < mu; ++nu) { stride *= g.L[nu]; phase_sum += x[nu]; }
    const double eta = (phase_sum & 1) ? -1.0 : 1.0;
    double f;
    int src_lex;
    if (!bwd) {
        f = 0.5 * eta * ((mu == 3 && x[3] == g.L[3] - 1) ? -1.0 : 1.0);
        src_lex = s.lex;
    } else {
        f = -0.5 * eta * ((mu == 3 && x[3] == 0) ? -1.0 : 1.0);
        src_lex = s.lex - stride + (x[mu] == 0 ? g.L[mu] * stride : 0);
    }
    const double *U = canon + ((size_t)src_lex * 4 + mu) * 18;
    double u[18], m[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) u[k] = U[k];

    if (RECON == 12 && !bwd) {
        // unitarity and determinant of the raw link (each link is the forward link of one site)
        double worst = 0.0;
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                double re = 0.0, im = 0.0;
#pragma unroll
                for (int k = 0; k < 3; ++k) {   // (U U^dag)_{ij} = sum_k U_ik conj(U_jk)
                    re += u[6 * i + 2 * k] * u[6 * j + 2 * k] + u[6 * i + 2 * k + 1] * u[6 * j + 2 * k + 1];
                    im += u[6 * i + 2 * k + 1] * u[6 * j + 2 * k] - u[6 * i + 2 * k] * u[6 * j + 2 * k + 1];
                }
                worst = fmax(worst, fmax(fabs(re - (i == j ? 1.0 : 0.0)), fabs(im)));
            }
        // det = row1 . (row2 x row3)
        double dr = 0.0, di = 0.0;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const int a = (j + 1) % 3, b = (j + 2) % 3;
            const double zr = u[6 + 2 * a] * u[12 + 2 * b] - u[6 + 2 * a + 1] * u[12 + 2 * b + 1]
                            - u[6 + 2 * b] * u[12 + 2 * a] + u[6 + 2 * b + 1] * u[12 + 2 * a + 1];
            const double zi = u[6 + 2 * a] * u[12 + 2 * b + 1] + u[6 + 2 * a + 1] * u[12 + 2 * b]
                            - u[6 + 2 * b] * u[12 + 2 * a + 1] - u[6 + 2 * b + 1] * u[12 + 2 * a];
            dr += u[2 * j] * zr - u[2 * j + 1] * zi;
            di += u[2 * j] * zi + u[2 * j + 1] * zr;
        }
        worst = fmax(worst, fmax(fabs(dr - 1.0), fabs(di)));
        if (!(worst <= 1e-12)) *reinterpret_cast<volatile int *>(not_su3) = 1;  // same value from all writers
    }

#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            if (!bwd) {
                m[6 * i + 2 * j] = f * u[6 * i + 2 * j];
                m[6 * i + 2 * j + 1] = f * u[6 * i + 2 * j + 1];
            } else {  // dagger
                m[6 * i + 2 * j] = f * u[6 * j + 2 * i];
                m[6 * i + 2 * j + 1] = -f * u[6 * j + 2 * i + 1];
            }
        }
    if constexpr (std::is_same<T, SplitTag>::value) {
        const size_t set = link_set_bytes<float, RECON>(g.Vh);
        write_planes_split<RECON>(packed + (size_t)blockIdx.y * set, 16 * set, g.Vh, e, m);
    } else {
        char *base = packed + (size_t)blockIdx.y * link_set_bytes<T, RECON>(g.Vh);
        write_planes<RECON>(base, g.Vh, e, m, T(0));
    }
}

template <typename T>
__global__ void __launch_bounds__(128)
vector_pack_kernel(const Geom g, const double *__restrict__ canon, char *__restrict__ v) {
    const int e = blockIdx.x * 128 + threadIdx.x;
    if (e >= g.Vh) return;
    T x[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) x[k] = (T)canon[(size_t)e * 6 + k];
    store_vec(v, g.Vh, e, x);
}

template <typename T>
__global__ void __launch_bounds__(128)
vector_unpack_kernel(const Geom g, const char *__restrict__ v, double *__restrict__ canon) {
    const int e = blockIdx.x * 128 + threadIdx.x;
    if (e >= g.Vh) return;
    T x[6];
    load_vec(v, g.Vh, e, x);
#pragma unroll
    for (int k = 0; k < 6; ++k) canon[(size_t)e * 6 + k] = (double)x[k];
}

}  // namespace stag

using namespace stag;

extern "C" int stag_gauge_load(const stag_ctx *ctx, const double *host_links,
                               double *dev_links_canonical, void *stream) {
    if (!ctx || !host_links || !dev_links_canonical) return STAG_ERR_BADARG;
    STAG_CUDA_OK(cudaMemcpyAsync(dev_links_canonical, host_links,
                                 stag_gauge_canonical_bytes(ctx), cudaMemcpyHostToDevice,
                                 static_cast<cudaStream_t>(stream)));
    return STAG_OK;
}

extern "C" int stag_gauge_pack(const stag_ctx *ctx, const double *dev_links_canonical,
                               void *dev_packed, int prec, int recon, void *stream) {
    if (!ctx || !dev_links_canonical || !dev_packed) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || !valid_recon(recon)) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Geom &g = ctx->g;
    const dim3 grid((g.Vh + 127) / 128, 16), block(128);
    char *out = static_cast<char *>(dev_packed);
    // recon 18 needs no host staging and stays asynchronous; recon 12 runs the SU(3) check, which writes a mapped
    // pinned status word of a staging slot leased for the duration of the call (and synchronises the stream)
    auto launch = [&](int *flag) {
        if (prec == STAG_F64_SPLIT) {
            if (recon == 18) gauge_pack_kernel<SplitTag, 18><<<grid, block, 0, st>>>(g, dev_links_canonical, out, flag);
            else gauge_pack_kernel<SplitTag, 12><<<grid, block, 0, st>>>(g, dev_links_canonical, out, flag);
        } else if (prec == STAG_F64) {
            if (recon == 18) gauge_pack_kernel<double, 18><<<grid, block, 0, st>>>(g, dev_links_canonical, out, flag);
            else gauge_pack_kernel<double, 12><<<grid, block, 0, st>>>(g, dev_links_canonical, out, flag);
        } else {
            if (recon == 18) gauge_pack_kernel<float, 18><<<grid, block, 0, st>>>(g, dev_links_canonical, out, flag);
            else gauge_pack_kernel<float, 12><<<grid, block, 0, st>>>(g, dev_links_canonical, out, flag);
        }
    };
    if (recon != 12) {
        launch(nullptr);
        STAG_CUDA_OK(cudaGetLastError());
        return STAG_OK;
    }
    SlotLease lease(ctx);
    int *host_flag = lease.slot().pinned_flags, *flag = nullptr;
    STAG_CUDA_OK(cudaHostGetDevicePointer((void **)&flag, host_flag, 0));
    host_flag[0] = 0;
    launch(flag);
    STAG_CUDA_OK(cudaGetLastError());
    STAG_CUDA_OK(cudaStreamSynchronize(st));
    if (host_flag[0] != 0) return STAG_ERR_NOT_SU3;
    return STAG_OK;
}

extern "C" int stag_vector_pack(const stag_ctx *ctx, const double *dev_canonical, void *dev_vec,
                                int prec, void *stream) {
    if (!ctx || !dev_canonical || !dev_vec || !valid_prec(prec)) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Geom &g = ctx->g;
    const int grid = (g.Vh + 127) / 128;
    if (prec != STAG_F32)
        vector_pack_kernel<double><<<grid, 128, 0, st>>>(g, dev_canonical, static_cast<char *>(dev_vec));
    else
        vector_pack_kernel<float><<<grid, 128, 0, st>>>(g, dev_canonical, static_cast<char *>(dev_vec));
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}

extern "C" int stag_vector_unpack(const stag_ctx *ctx, const void *dev_vec, int prec,
                                  double *dev_canonical, void *stream) {
    if (!ctx || !dev_canonical || !dev_vec || !valid_prec(prec)) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Geom &g = ctx->g;
    const int grid = (g.Vh + 127) / 128;
    if (prec != STAG_F32)
        vector_unpack_kernel<double><<<grid, 128, 0, st>>>(g, static_cast<const char *>(dev_vec), dev_canonical);
    else
        vector_unpack_kernel<float><<<grid, 128, 0, st>>>(g, static_cast<const char *>(dev_vec), dev_canonical);
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}
