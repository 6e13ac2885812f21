// zda_density_vjp_static (include/zda.h): the density map's VJP (a2 transposed: PAPER.md:72-76 Eq. 6, :83 filter and
// projection; R13, R14) for callers that must not allocate.  It is the dF_drho tail of zda_gradient
// (zda_zone_impl.cuh Zone::gradient) with the same kernels in the same order; the only difference is where the two
// intermediate planes live: there in the zone's workspace, here in ONE file-scope device array that every call shares.
//
// No cudaMalloc / cudaFree / allocating library routine anywhere in this file, no host heap either (the filter weights
// sit on the stack).  The one piece of set-up, once per device with that device current, is cudaGetSymbolAddress:
// in HOST code the array's name is a host-side stand-in, not a device address, so kernels get the looked-up pointer.
#include <cmath>
#include <mutex>
#include "zda_zone_impl.cuh"

namespace zda {

static_assert(ZDA_STATIC_SCRATCH_BYTES % 512 == 0, "two planes, each a multiple of 256 B");
// Held by every GPU that loads libzda.so until the process exits.  Contents survive from call to call.
static __device__ __align__(256) unsigned char g_static_scratch[ZDA_STATIC_SCRATCH_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
static std::mutex g_static_mu;
static unsigned char* g_static_ptr[STATIC_MAX_DEVICES];   // device address of g_static_scratch, per device ordinal

// Device address of the scratch array on the CURRENT device (looked up once per device).
static int static_scratch(unsigned char** out) {
    int dev = -1;
    ZDA_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(ZDA_E_BADARG, "device ordinal %d outside 0..%d", dev, STATIC_MAX_DEVICES - 1);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        ZDA_CUDA_OK(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return fail(ZDA_E_CUDA, "cudaGetSymbolAddress gave %p for the static scratch", p);
        g_static_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_ptr[dev];
    return ZDA_OK;
}

// the Gaussian weights exactly as Zone::filter_weights builds them (double, normalised, rounded once), on the stack
template <class R> static FilterW<R> static_filter_weights(double sigma) {
    FilterW<R> W;
    W.Rad = (int)std::ceil(3.0 * sigma);
    double w[2 * MAX_FILTER_R + 1], sum = 0.0;
    for (int t = -W.Rad; t <= W.Rad; ++t) { w[t + W.Rad] = std::exp(-0.5 * (t / sigma) * (t / sigma)); sum += w[t + W.Rad]; }
    for (int t = 0; t <= 2 * W.Rad; ++t) W.w[t] = (R)(w[t] / sum);
    for (int t = 2 * W.Rad + 1; t <= 2 * MAX_FILTER_R; ++t) W.w[t] = R(0);
    return W;
}

template <class R>
static int density_vjp_static(int Nrd, int Nphi, const void* rho, const void* gz, void* out, double eps0, double eps_h,
                              double sigma, double beta, double eta, cudaStream_t st) {
    const size_t n2 = (size_t)Nrd * Nphi;
    const size_t plane = (n2 * sizeof(R) + 255) & ~size_t(255);
    if (2 * plane > (size_t)ZDA_STATIC_SCRATCH_BYTES)
        return fail(ZDA_E_BADARG, "zda_density_vjp_static: Nr_d x Nphi = %d x %d needs %zu B of scratch, the static array holds %zu B "
                                  "(at most %zu cells in this precision); use zda_gradient, whose scratch is in the caller's workspace",
                    Nrd, Nphi, 2 * plane, (size_t)ZDA_STATIC_SCRATCH_BYTES, (size_t)ZDA_STATIC_SCRATCH_BYTES / 2 / sizeof(R));
    unsigned char* base = nullptr;
    int rc = static_scratch(&base);
    if (rc != ZDA_OK) return rc;
    R* s0 = reinterpret_cast<R*>(base);
    R* s1 = reinterpret_cast<R*>(base + plane);
    const FilterW<R> W = static_filter_weights<R>(sigma);
    const dim3 grid((Nrd + 127) / 128, Nphi);
    // forward filter (r, then phi): rho_f, which the projection derivative is taken at.  Every scratch element a kernel
    // reads was written earlier in THIS call (whole planes each time), so nothing has to start at zero.
    filter_r_kernel<R><<<grid, 128, 0, st>>>((const R*)rho, s0, Nrd, Nphi, W);
    filter_phi_kernel<R><<<grid, 128, 0, st>>>(s0, s1, Nrd, Nphi, W);
    // x (eps_h - eps0) x d rho_bar / d rho_f, then the transposed filter (phi first, then r)
    project_vjp_kernel<R><<<(int)((n2 + 255) / 256), 256, 0, st>>>((const R*)gz, s1, s0, (int)n2, (R)eps0, (R)eps_h, (R)beta, (R)eta);
    filter_phi_kernel<R><<<grid, 128, 0, st>>>(s0, s1, Nrd, Nphi, W);
    filter_r_T_kernel<R><<<grid, 128, 0, st>>>(s1, (R*)out, Nrd, Nphi, W);
    ZDA_CUDA_OK(cudaGetLastError());
    return ZDA_OK;
}

}  // namespace zda

using namespace zda;

extern "C" int zda_density_vjp_static(int precision, int Nr_d, int Nphi, const void* rho2d, const void* dF_deps_zsum, void* dF_drho,
                                      double eps0, double eps_h, double filt_sigma, double beta, double eta, void* stream) {
    if (precision != 32 && precision != 64) return fail(ZDA_E_BADARG, "precision must be 32 or 64");
    if (!rho2d || !dF_deps_zsum || !dF_drho) return fail(ZDA_E_BADARG, "rho2d, dF_deps_zsum and dF_drho must be device pointers, not NULL");
    if (Nr_d < 1 || Nphi < 1 || Nphi > 65535) return fail(ZDA_E_BADARG, "need Nr_d >= 1 and 1 <= Nphi <= 65535");
    if (!(eps0 > 0 && eps_h > 0)) return fail(ZDA_E_BADARG, "eps0, eps_h must be > 0");
    if (!(filt_sigma > 0) || std::ceil(3.0 * filt_sigma) > MAX_FILTER_R) return fail(ZDA_E_BADARG, "filt_sigma must be in (0, 16]");
    if (!(beta > 0) || !(eta > 0 && eta < 1)) return fail(ZDA_E_BADARG, "need beta > 0 and 0 < eta < 1");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    try {   // nothing throws across the ABI (the mutex is the only thing here that could)
        if (precision == 32) return density_vjp_static<float>(Nr_d, Nphi, rho2d, dF_deps_zsum, dF_drho, eps0, eps_h, filt_sigma, beta, eta, st);
        return density_vjp_static<double>(Nr_d, Nphi, rho2d, dF_deps_zsum, dF_drho, eps0, eps_h, filt_sigma, beta, eta, st);
    } catch (...) {
        return fail(ZDA_E_BADARG, "zda_density_vjp_static: unexpected exception");
    }
}
