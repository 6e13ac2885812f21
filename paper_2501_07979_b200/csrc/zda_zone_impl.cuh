// Zone implementation for one floating-point type (instantiated in zda_f32.cu, zda_f64.cu).
// Host orchestration + the small kernels around the time loop: material maps (a2), adjoint
// source builder (a7), objective, gradient (a9).  The time-loop kernels are in
// zda_kernels_split.cuh and zda_kernels_fused.cuh.
#pragma once
#include <cmath>
#include <cstring>
#include <vector>
#include "zda_common.h"
#include "zda_device.cuh"
#include "zda_kernels_split.cuh"
#include "zda_kernels_fused.cuh"
#include "zda_kernels_fused2.cuh"

namespace zda {

// ---------------------------------------------------------------------------------------------
// small kernels
// ---------------------------------------------------------------------------------------------
constexpr int MAX_FILTER_R = 48;
template <class R> struct FilterW { int Rad; R w[2 * MAX_FILTER_R + 1]; };

// cE = dt / eps on the design box (R3); eps dense [kd][j][id] -> cE [kd][j][pitch] at i = di0 + id
template <class R>
__global__ void eps_to_cE_kernel(const R* __restrict__ eps, R* __restrict__ cE, int Nrd, int Nphi, int Ld,
                                 int pitch, int di0, R dt) {
    const size_t n = (size_t)Nrd * Nphi * Ld;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const int id = (int)(t % Nrd);
        const size_t rowi = t / Nrd;   // kd * Nphi + j
        cE[rowi * pitch + di0 + id] = dt / eps[t];
    }
}

// cE = background dt / eps(z) on every material plane [Lm][Nphi][pitch] (zone creation: the design box starts as background)
template <class R>
__global__ void fill_cE_bg_kernel(R* __restrict__ cE, const R* __restrict__ zc, int Nz, int mk0, int Lm, size_t plane) {
    const size_t n = (size_t)Lm * plane;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x)
        cE[t] = zc[ZC_CE_BG * Nz + mk0 + (int)(t / plane)];
}

// per-voxel eps over the whole zone (zda_set_eps_volume): eps dense [k][j][i] -> cE [k][j][pitch]
template <class R>
__global__ void eps_volume_to_cE_kernel(const R* __restrict__ eps, R* __restrict__ cE, int Nr, size_t rows, int pitch, R dt) {
    const size_t n = rows * Nr;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x)
        cE[(t / Nr) * pitch + (t % Nr)] = dt / eps[t];
}

// cE_axis[k] = dt / mean_j eps[0, j, k] (R4); eps = dt / cE
template <class R>
__global__ void axis_cE_kernel(const R* __restrict__ cE_design, const R* __restrict__ zc, R* __restrict__ cE_axis,
                               int Nz, int Nphi, int pitch, int mk0, int mk1, R dt) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= Nz) return;
    if (!(k >= mk0 && k < mk1)) { cE_axis[k] = zc[ZC_CE_BG * Nz + k]; return; }
    R sum = 0;
    for (int j = 0; j < Nphi; ++j) sum += dt / cE_design[((size_t)(k - mk0) * Nphi + j) * pitch];
    cE_axis[k] = dt / (sum / R(Nphi));
}

// a2, filter along r (edge-clamped): out[j][i] = sum_d w[d] in[j][clamp(i + d)]
template <class R>
__global__ void filter_r_kernel(const R* __restrict__ in, R* __restrict__ out, int Nrd, int Nphi, const FilterW<R> W) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= Nrd) return;
    R acc = 0;
    for (int d = -W.Rad; d <= W.Rad; ++d) {
        int ii = i + d; ii = ii < 0 ? 0 : (ii > Nrd - 1 ? Nrd - 1 : ii);
        acc += W.w[d + W.Rad] * in[(size_t)j * Nrd + ii];
    }
    out[(size_t)j * Nrd + i] = acc;
}
// filter along phi (periodic): out[j][i] = sum_d w[d] in[(j + d) mod Nphi][i]
template <class R>
__global__ void filter_phi_kernel(const R* __restrict__ in, R* __restrict__ out, int Nrd, int Nphi, const FilterW<R> W) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= Nrd) return;
    R acc = 0;
    for (int d = -W.Rad; d <= W.Rad; ++d) {
        int jj = (j + d) % Nphi; if (jj < 0) jj += Nphi;
        acc += W.w[d + W.Rad] * in[(size_t)jj * Nrd + i];
    }
    out[(size_t)j * Nrd + i] = acc;
}
// transpose of filter_r (scatter into clamp(i + d), written as a gather)
template <class R>
__global__ void filter_r_T_kernel(const R* __restrict__ in, R* __restrict__ out, int Nrd, int Nphi, const FilterW<R> W) {
    const int ii = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (ii >= Nrd) return;
    const R* row = in + (size_t)j * Nrd;
    R acc = 0;
    for (int d = -W.Rad; d <= W.Rad; ++d) {          // sources i = ii - d that land on ii unclamped
        const int i = ii - d;
        if (i >= 0 && i < Nrd) acc += W.w[d + W.Rad] * row[i];
    }
    if (ii == 0)                                      // sources clamped to the low edge: i + d < 0
        for (int i = 0; i < W.Rad && i < Nrd; ++i)
            for (int d = -W.Rad; d < -i; ++d) acc += W.w[d + W.Rad] * row[i];
    if (ii == Nrd - 1)                                // sources clamped to the high edge: i + d > Nrd - 1
        for (int i = (Nrd - W.Rad > 0 ? Nrd - W.Rad : 0); i < Nrd; ++i)
            for (int d = Nrd - i; d <= W.Rad; ++d) acc += W.w[d + W.Rad] * row[i];
    out[(size_t)j * Nrd + ii] = acc;
}

// R22: the paper's conic filter in the physical (r, r phi) metric.  Cell (i, j) sits at
// r_i = r_first + i dr; d^2 = (a dr)^2 + (rbar b dphi)^2 with rbar = (r_i + r_{i+a})/2, w = max(0, 1 - d/R), all
// periodic images b (cell (j + b) mod Nphi), r truncated at the region's edges.
//   MODE 0: out = sum w in / sum w   (the filter)
//   MODE 1: out = in / sum w         (first half of the transpose)
//   MODE 2: out = sum w in           (second half: the un-normalised stencil is symmetric)
template <class R> struct ConicP { R r_first, dr, dphi, inv_R; int a_max, b_max; };
template <class R, int MODE>
__global__ void conic_kernel(const R* __restrict__ in, R* __restrict__ out, int Nrd, int Nphi, const ConicP<R> C) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= Nrd) return;
    const R ri = C.r_first + R(i) * C.dr;
    R acc = 0, norm = 0;
    for (int a = -C.a_max; a <= C.a_max; ++a) {
        const int ii = i + a;
        if (ii < 0 || ii >= Nrd) continue;
        const R rbar = R(0.5) * (ri + (C.r_first + R(ii) * C.dr));
        const R da = R(i - ii) * C.dr;
        int jj = (j - C.b_max) % Nphi; if (jj < 0) jj += Nphi;
        for (int b = -C.b_max; b <= C.b_max; ++b) {
            const R db = rbar * R(b) * C.dphi;
            const R w = R(1) - sqrt(da * da + db * db) * C.inv_R;
            if (w > R(0)) {
                norm += w;
                if (MODE != 1) acc += w * in[(size_t)jj * Nrd + ii];
            }
            if (++jj == Nphi) jj = 0;
        }
    }
    out[(size_t)j * Nrd + i] = MODE == 0 ? acc / norm : (MODE == 1 ? in[(size_t)j * Nrd + i] / norm : acc);
}

// projection (R13) + Eq. 6 + extrusion (R14): writes cE = dt / eps for every layer
template <class R>
__global__ void project_extrude_kernel(const R* __restrict__ rho_f, R* __restrict__ cE, int Nrd, int Nphi, int Ld,
                                       int pitch, int di0, R dt, R eps0, R eps_h, R beta, R eta) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (id >= Nrd) return;
    const R den = tanh(beta * eta) + tanh(beta * (R(1) - eta));
    const R rb = (tanh(beta * eta) + tanh(beta * (rho_f[(size_t)j * Nrd + id] - eta))) / den;
    const R eps = eps0 + rb * (eps_h - eps0);
    const R c = dt / eps;
    for (int kd = 0; kd < Ld; ++kd) cE[((size_t)kd * Nphi + j) * pitch + di0 + id] = c;
}
// VJP step: g2d <- g_zsum (eps_h - eps0) d rho_bar / d rho_f
template <class R>
__global__ void project_vjp_kernel(const R* __restrict__ gz, const R* __restrict__ rho_f, R* __restrict__ out,
                                   int n, R eps0, R eps_h, R beta, R eta) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const R den = tanh(beta * eta) + tanh(beta * (R(1) - eta));
    const R th = tanh(beta * (rho_f[t] - eta));
    out[t] = gz[t] * (eps_h - eps0) * (beta * (R(1) - th * th) / den);
}

// warp-shuffle + shared-memory block reduction of doubles
__device__ __forceinline__ double block_reduce_sum(double v) {
    __shared__ double sm[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sm[w] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? sm[threadIdx.x] : 0.0;
    if (w == 0) for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// R9: F = sum_f sum_{c in r,phi} sum_{i in mask, j} W_c(i) |Ehat_{c,f}(i, j, k_m)|^2; partial sums per block
template <class R>
__global__ void objective_kernel(const Cx<R>* __restrict__ mon, const R* __restrict__ rc, double* __restrict__ partial,
                                 int Nr, int Nphi, int pitch, int F, int m0, int m1) {
    const size_t plane = (size_t)pitch * Nphi;
    double acc = 0.0;
    const size_t n = (size_t)F * 2 * plane;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % pitch);
        if (i < m0 || i >= m1) continue;
        const size_t fc = t / plane;            // f * 2 + c
        const int f = (int)(fc / 2), c = (int)(fc % 2);
        const Cx<R> v = mon[((size_t)f * 3 + c) * plane + (t % plane)];
        const R w = rc[(c == 0 ? RC_W_HALF : RC_W_INT) * pitch + i];
        acc += (double)w * ((double)v.x * v.x + (double)v.y * v.y);
    }
    acc = block_reduce_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
}

// R20: S_f = sum_{c in r,phi} sum_{i in mask, j} g_{c,f}(i,j) Ehat_{c,f}(i,j,k_m); block (b, f) writes its partial
// (re, im) to partial[(f * gridDim.x + b) * 2 ..]; g lives in the planes (f*3 + c) of a monitor-shaped array
template <class R>
__global__ void focal_sum_kernel(const Cx<R>* __restrict__ mon, const Cx<R>* __restrict__ gw, double* __restrict__ partial,
                                 int Nphi, int pitch, int m0, int m1) {
    const size_t plane = (size_t)pitch * Nphi;
    const int f = blockIdx.y;
    double re = 0.0, im = 0.0;
    for (int c = 0; c < 2; ++c) {
        const size_t base = ((size_t)f * 3 + c) * plane;
        for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < plane; t += (size_t)gridDim.x * blockDim.x) {
            const int i = (int)(t % pitch);
            if (i < m0 || i >= m1) continue;
            const Cx<R> v = mon[base + t], w = gw[base + t];
            re += (double)w.x * v.x - (double)w.y * v.y;
            im += (double)w.x * v.y + (double)w.y * v.x;
        }
    }
    re = block_reduce_sum(re);
    __syncthreads();
    im = block_reduce_sum(im);
    if (threadIdx.x == 0) {
        partial[((size_t)f * gridDim.x + blockIdx.x) * 2] = re;
        partial[((size_t)f * gridDim.x + blockIdx.x) * 2 + 1] = im;
    }
}

// R24 (include/zda.h zda_build_focal_weights): the wedge sums of the x-polarisation factors,
//   C[j] = sum_{w < n} p^w cos(phi_j + w tau),   C[Nphi + j] = -sum_{w < n} p^w sin(phi_{j+1/2} + w tau)
// (E_x = E_r cos(phi) - E_phi sin(phi); the other wedges carry the Bloch-continued field), in double; p^w by repeated
// multiplication, w ascending.
template <class R>   // (R only keeps the two precision units' instances apart)
__global__ void wedge_sum_kernel(Cx<double>* __restrict__ C, int Nphi, int n, double dphi, double tau, double p_re, double p_im) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Nphi) return;
    double cr = 0, ci = 0, sr = 0, si = 0, pr = 1, pi = 0;
    for (int w = 0; w < n; ++w) {
        const double c0 = cos(j * dphi + w * tau), s0 = sin((j + 0.5) * dphi + w * tau);
        cr += pr * c0; ci += pi * c0; sr += pr * s0; si += pi * s0;
        const double nr = pr * p_re - pi * p_im, ni = pr * p_im + pi * p_re;
        pr = nr; pi = ni;
    }
    C[j] = Cx<double>{cr, ci};
    C[Nphi + j] = Cx<double>{-sr, -si};
}
// g[f][c][j][i] = h_f(rho) rho dr dphi C_c[j],  h = -(1 / 2 pi) (i k - 1 / R) exp(i k R) dz / R^2 (first Rayleigh-Sommerfeld
// integral to the on-axis point dz above the plane), rho = r_{i+1/2} (c = 0) or r_i (c = 1); everything in double, rounded
// once; written into planes (f*3 + c) of the monitor-shaped weight array.
template <class R> struct FocalK { int F; double k[ZDA_MAX_FREQ]; };
template <class R>
__global__ void focal_weights_kernel(const Cx<double>* __restrict__ C, Cx<R>* __restrict__ g, int Nr, int Nphi, int pitch,
                                     double r_in, double dr, double dA, double dz, const FocalK<R> K) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= Nr) return;
    const size_t plane = (size_t)pitch * Nphi;
    for (int c = 0; c < 2; ++c) {
        const double rho = r_in + (i + (c == 0 ? 0.5 : 0.0)) * dr;
        const double Rr = sqrt(rho * rho + dz * dz);
        const Cx<double> b = C[(size_t)c * Nphi + j];
        for (int f = 0; f < K.F; ++f) {
            const double k = K.k[f];
            const double er = cos(k * Rr), ei = sin(k * Rr);
            const double ar = -1.0 / Rr, ai = k;                                   // (i k - 1 / R)
            const double s = -(1.0 / 6.283185307179586476925286766559) * dz / (Rr * Rr) * rho * dA;
            const Cx<double> a{s * (ar * er - ai * ei), s * (ar * ei + ai * er)};
            g[((size_t)f * 3 + c) * plane + (size_t)j * pitch + i] = Cx<R>{(R)(a.x * b.x - a.y * b.y), (R)(a.x * b.y + a.y * b.x)};
        }
    }
}

// a7 (R11): per monitor-plane point, the prescribed half-step DTFT a_f (0 outside the mask):
//   monitor energy (gw == nullptr): a_f = conj(Ehat^fwd_{c,f});
//   focal intensity (R20):          a_f = coef[f] g_{c,f} / W_c(i), coef[f] = u_f conj(S_f);
// then A_q = sum_col Minv[q][col] rhs[col].
// real fields:    rhs = [Re a_0.., Im a_0..] (2F), A_q real, q < 2F
// complex fields: A_f = sum_f' Vinv[f][f'] a_f' (complex), Minv holds Re then Im parts
template <class R> struct FocalCoef { Cx<R> c[ZDA_MAX_FREQ]; };
template <class T>
__global__ void adjoint_source_kernel(const Cx<typename ElemTraits<T>::Real>* __restrict__ mon, T* __restrict__ A_r,
                                      T* __restrict__ A_phi, const typename ElemTraits<T>::Real* __restrict__ Minv,
                                      int Nr, int Nphi, int pitch, int F, int m0, int m1,
                                      const Cx<typename ElemTraits<T>::Real>* __restrict__ gw,
                                      const typename ElemTraits<T>::Real* __restrict__ rc,
                                      const FocalCoef<typename ElemTraits<T>::Real> coef) {
    using R = typename ElemTraits<T>::Real;
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= pitch) return;
    const size_t plane = (size_t)pitch * Nphi, pj = (size_t)j * pitch + i;
    const bool live = (i >= m0 && i < m1 && i < Nr);
    for (int c = 0; c < 2; ++c) {
        T* A = c == 0 ? A_r : A_phi;
        Cx<R> a[ZDA_MAX_FREQ];
        if (gw) {
            const R w = rc[(c == 0 ? RC_W_HALF : RC_W_INT) * pitch + i];
            const R iw = w > R(0) ? R(1) / w : R(0);
            for (int f = 0; f < F; ++f) {
                const Cx<R> v = cmul(coef.c[f], gw[((size_t)f * 3 + c) * plane + pj]);
                a[f] = live ? Cx<R>{v.x * iw, v.y * iw} : Cx<R>{R(0), R(0)};
            }
        } else {
            for (int f = 0; f < F; ++f) {
                const Cx<R> v = mon[((size_t)f * 3 + c) * plane + pj];
                a[f] = live ? Cx<R>{v.x, -v.y} : Cx<R>{R(0), R(0)};
            }
        }
        if constexpr (ElemTraits<T>::cplx) {
            for (int q = 0; q < F; ++q) {
                Cx<R> acc{R(0), R(0)};
                for (int f = 0; f < F; ++f) acc = acc + cmul(Cx<R>{Minv[q * F + f], Minv[F * F + q * F + f]}, a[f]);
                A[(size_t)q * plane + pj] = acc;
            }
        } else {
            const int n2 = 2 * F;
            for (int q = 0; q < n2; ++q) {
                R acc = 0;
                for (int f = 0; f < F; ++f) acc += Minv[q * n2 + f] * a[f].x;
                for (int f = 0; f < F; ++f) acc += Minv[q * n2 + F + f] * a[f].y;
                A[(size_t)q * plane + pj] = acc;
            }
        }
    }
}

// a9 (R9-R12): dF/deps = sum_f sum_c 2 Re[(-i Omega_f) W_c(i) Ehat^fwd Ehat^adj] = sum 2 Omega_f W_c Im(fwd adj);
// one thread per (id, j), serial over the layer so that the z-sum stays in a register.
template <class R> struct GradParams { int F; R Omega[ZDA_MAX_FREQ]; };
template <class R>
__global__ void gradient_kernel(const Cx<R>* __restrict__ fwd, const Cx<R>* __restrict__ adj, const R* __restrict__ rc,
                                R* __restrict__ g_box, R* __restrict__ g_zsum, int Nrd, int Nphi, int Ld, int pitch,
                                int di0, const GradParams<R> G) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (id >= Nrd) return;
    const int i = di0 + id;
    const size_t plane = (size_t)pitch * Nphi, pj = (size_t)j * pitch + i;
    const R W[3] = {rc[RC_W_HALF * pitch + i], rc[RC_W_INT * pitch + i], rc[RC_W_Z * pitch + i]};
    R zsum = 0;
    for (int kd = 0; kd < Ld; ++kd) {
        R g = 0;
        for (int f = 0; f < G.F; ++f)
            for (int c = 0; c < 3; ++c) {
                const size_t o = (((size_t)f * 3 + c) * Ld + kd) * plane + pj;
                const Cx<R> a = fwd[o], b = adj[o];
                g += R(2) * (G.Omega[f] * W[c]) * (a.x * b.y + a.y * b.x);
            }
        if (g_box) g_box[((size_t)kd * Nphi + j) * Nrd + id] = g;
        zsum += g;
    }
    if (g_zsum) g_zsum[(size_t)j * Nrd + id] = zsum;
}

// a6, accumulators of the design box visited every s steps: Ehat_{c,f} <- (..((Ehat + tw_{n0} E^{n0+1}) +
// tw_{n0+1} E^{n0+2}) ..) + tw_{n0+m-1} E^{n0+m}, the terms in step order exactly as the every-step update adds them.
// Source t is a design-layer copy kept by the fused kernel (ring slot) or one of the two time buffers of the field.
constexpr int DFT_MAX_PERIOD = 8;
template <class T> struct VisitSrc { const T* p[3]; size_t kstride; };
template <class T> struct VisitParams {
    using R = typename ElemTraits<T>::Real;
    int m, F, n0, Nphi, Ld, pitch, di0, di1;
    size_t plane;
    VisitSrc<T> src[DFT_MAX_PERIOD];
    Cx<R>* dft;
    const Cx<R>* tw;
};
// One thread per 16-byte group of E along r (4 float / 2 complex-float or double / 1 complex-double), like the fused
// kernel: whole groups are read and written; entries of a group outside the design box are scratch nothing reads (the ring
// copies and the accumulators hold whole groups for the same reason).
template <class T>
__global__ void __launch_bounds__(128) dft_visit_kernel(const __grid_constant__ VisitParams<T> V) {
    using R = typename ElemTraits<T>::Real;
    constexpr int VEC = VecT<T>::N;
    using DV = DftV<R, VEC>;
    const int ig = (V.di0 / VEC + blockIdx.x * 128 + threadIdx.x) * VEC, j = blockIdx.y, kd = blockIdx.z;
    if (ig >= V.di1) return;
    const size_t rowo = (size_t)j * V.pitch + ig;
    VecT<T> e[DFT_MAX_PERIOD][3];
#pragma unroll
    for (int t = 0; t < DFT_MAX_PERIOD; ++t)
        if (t < V.m) {
#pragma unroll
            for (int c = 0; c < 3; ++c) e[t][c] = ldg_vec(V.src[t].p[c] + (size_t)kd * V.src[t].kstride + rowo);
        }
    const size_t cstride = (size_t)V.Ld * V.plane;
    for (int f = 0; f < V.F; ++f) {
        Cx<R>* d = V.dft + ((size_t)f * 3 * V.Ld + kd) * V.plane + rowo;
        DV a0 = *reinterpret_cast<const DV*>(d), a1 = *reinterpret_cast<const DV*>(d + cstride),
           a2 = *reinterpret_cast<const DV*>(d + 2 * cstride);
#pragma unroll
        for (int t = 0; t < DFT_MAX_PERIOD; ++t)
            if (t < V.m) {
                const Cx<R> tw = V.tw[(size_t)(V.n0 + t) * V.F + f];
#pragma unroll
                for (int q = 0; q < VEC; ++q) {
                    a0.v[q] = a0.v[q] + tw_mul(tw, e[t][0].v[q]);
                    a1.v[q] = a1.v[q] + tw_mul(tw, e[t][1].v[q]);
                    a2.v[q] = a2.v[q] + tw_mul(tw, e[t][2].v[q]);
                }
            }
        *reinterpret_cast<DV*>(d) = a0;
        *reinterpret_cast<DV*>(d + cstride) = a1;
        *reinterpret_cast<DV*>(d + 2 * cstride) = a2;
    }
}

// failure detector: count of non-finite E values
template <class T>
__global__ void nonfinite_kernel(const T* __restrict__ a, size_t n, double* __restrict__ partial) {
    double acc = 0.0;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        if constexpr (ElemTraits<T>::cplx) acc += (isfinite(a[t].x) && isfinite(a[t].y)) ? 0.0 : 1.0;
        else acc += isfinite(a[t]) ? 0.0 : 1.0;
    }
    acc = block_reduce_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
}

// in-run failure detector (ZDA_OPT_CHECK_EVERY): raises *flag when the array holds a non-finite value
template <class T>
__global__ void nonfinite_flag_kernel(const T* __restrict__ a, size_t n, int* __restrict__ flag) {
    bool bad = false;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        if constexpr (ElemTraits<T>::cplx) bad = bad || !(isfinite(a[t].x) && isfinite(a[t].y));
        else bad = bad || !isfinite(a[t]);
    }
    if (bad) atomicOr(flag, 1);
}

// ---------------------------------------------------------------------------------------------
// the zone
// ---------------------------------------------------------------------------------------------
template <class R> struct ZoneLayout {
    // device arrays carved from the workspace; es = element size of a field (R or Cx<R>)
    char* E[2][3];  char* H[2][3];   // [Nz][Nphi + 2 FIELD_GHOST][pitch] each; the 12 arrays are equally spaced (fstride)
    char* fbase; size_t fstride;     // array a = b * 6 + (E ? c : 3 + c) starts at fbase + a * fstride
    char* psiH_z[2][2]; char* psiH_r[2][2]; char* psiE_z[2][2]; char* psiE_r[2][2];   // [time buffer][component]
    char* chiH[2][2]; char* chiE[2][2];   // R25 (rpml_exact): auxiliaries of the 1/r~ operator, r-slab layout
    R* rc; R* zc; R* cE_design;
    char* axis_mean;
    Cx<R>* dft_design[2]; Cx<R>* dft_mon[2];
    char* A[2][2];          // [fwd/adj][r/phi] sheets, cap_terms planes each
    char* s_tab[2];         // [fwd/adj] tables, cap_terms x max_steps
    Cx<R>* tw;              // max_steps x F
    R* rho; R* rho_f; R* tmp2d; R* g2d;   // density map scratch (Nrd x Nphi)
    R* staging;             // design-box sized scratch (dense), also used for host<->device staging
    R* Minv;                // adjoint-source matrix
    double* partial;        // reduction scratch (1024)
    int* step_counter;      // device-side step index of the graph-replayed split path
    char* ring;             // (ring_period - 2) design-layer copies of E, [slot][3][Ld][Nphi][pitch] field elements
    int ring_period;        // the visit period the ring was carved for (2: no ring); runs may use any period <= it
    size_t state_begin, state_end;   // byte range holding fields + psi (zeroed by reset)
};

constexpr int N_PARTIAL = 1024;

// How often the design-box accumulators are visited when the fused kernel runs (2 = inside the kernel, every second
// launch; 4 or 8 = by dft_visit_kernel).  Bytes per design voxel and step: the accumulators cost 48 F / s (read + write),
// every E copy 3 es: s = 2 re-reads one step from the other time buffer ((48 F + 3 es) / 2); s > 2 reads all s steps and
// has written s - 2 of them to the ring ((48 F + 3 es (2 s - 2)) / s).  The cheapest of 2, 4, 8 is taken: many
// frequencies favour long periods (config 4, F = 6 real: 150 -> 57 B), one frequency keeps s = 2.
inline int dft_visit_period(const zda_zone_desc& d) {
    if (d.has_axis) return 2;     // split path
    const double rb = d.precision == 64 ? 8.0 : 4.0;
    const double acc = 12.0 * rb * d.n_freq, ec = 3.0 * (d.complex_fields ? 2 : 1) * rb;
    int best = 2;
    double cost = (acc + ec) / 2.0;
    for (int sp : {4, 8}) {
        const double c = (acc + ec * (2 * sp - 2)) / sp;
        if (c < 0.9 * cost) { best = sp; cost = c; }
    }
    return best;
}

template <class R>
static void carve(const zda_zone_desc& d, int max_steps, int pitch, Arena& ar, ZoneLayout<R>& L) {
    const size_t es = d.complex_fields ? 2 * sizeof(R) : sizeof(R);
    const size_t plane = (size_t)pitch * d.Nphi;
    const size_t fvol = (size_t)pitch * (d.Nphi + 2 * field_ghost(d)) * d.Nz;
    const int npz = d.npml_z_lo + d.npml_z_hi, npr = d.npml_r_lo + d.npml_r_hi;
    const int Ld = d.design_k1 - d.design_k0, Nrd = d.design_i1 - d.design_i0, F = d.n_freq;
    const int cap_terms = std::max(2, d.complex_fields ? F : 2 * F);
    ar.off = (ar.off + 255) & ~size_t(255);
    L.state_begin = ar.off;
    L.fstride = (fvol * es + 255) & ~size_t(255);
    L.fbase = ar.take<char>(12 * L.fstride);
    for (int b = 0; b < 2; ++b)
        for (int c = 0; c < 3; ++c) {
            L.E[b][c] = L.fbase ? L.fbase + (size_t)(b * 6 + c) * L.fstride : nullptr;
            L.H[b][c] = L.fbase ? L.fbase + (size_t)(b * 6 + 3 + c) * L.fstride : nullptr;
        }
    for (int b = 0; b < 2; ++b)
        for (int c = 0; c < 2; ++c) {
            L.psiH_z[b][c] = ar.take<char>((size_t)std::max(npz, 1) * plane * es);
            L.psiH_r[b][c] = ar.take<char>((size_t)d.Nz * d.Nphi * std::max(npr, 1) * es);
        }
    for (int b = 0; b < 2; ++b)
        for (int c = 0; c < 2; ++c) {
            L.psiE_z[b][c] = ar.take<char>((size_t)std::max(npz, 1) * plane * es);
            L.psiE_r[b][c] = ar.take<char>((size_t)d.Nz * d.Nphi * std::max(npr, 1) * es);
        }
    for (int b = 0; b < 2; ++b)
        for (int c = 0; c < 2; ++c) {
            L.chiH[b][c] = d.rpml_exact ? ar.take<char>((size_t)d.Nz * d.Nphi * std::max(npr, 1) * es) : nullptr;
            L.chiE[b][c] = d.rpml_exact ? ar.take<char>((size_t)d.Nz * d.Nphi * std::max(npr, 1) * es) : nullptr;
        }
    L.axis_mean = ar.take<char>((size_t)d.Nz * es);
    ar.off = (ar.off + 255) & ~size_t(255);
    L.state_end = ar.off;
    L.rc = ar.take<R>((size_t)RC_COUNT * pitch);
    L.zc = ar.take<R>((size_t)ZC_COUNT * d.Nz);
    L.cE_design = ar.take<R>((size_t)(d.eps_volume ? d.Nz : Ld) * plane);
    for (int w = 0; w < 2; ++w) {
        L.dft_design[w] = ar.take<Cx<R>>((size_t)F * 3 * Ld * plane);
        L.dft_mon[w] = ar.take<Cx<R>>((size_t)F * 3 * plane);
        for (int c = 0; c < 2; ++c) L.A[w][c] = ar.take<char>((size_t)cap_terms * plane * es);
        L.s_tab[w] = ar.take<char>((size_t)cap_terms * max_steps * es);
    }
    L.tw = ar.take<Cx<R>>((size_t)max_steps * F);
    L.rho = ar.take<R>((size_t)Nrd * d.Nphi);
    L.rho_f = ar.take<R>((size_t)Nrd * d.Nphi);
    L.tmp2d = ar.take<R>((size_t)Nrd * d.Nphi);
    L.g2d = ar.take<R>((size_t)Nrd * d.Nphi);
    L.staging = ar.take<R>((size_t)Nrd * d.Nphi * Ld);
    L.Minv = ar.take<R>(4 * ZDA_MAX_FREQ * ZDA_MAX_FREQ);
    L.partial = ar.take<double>(N_PARTIAL);
    L.step_counter = ar.take<int>(64);
    ar.off = (ar.off + 255) & ~size_t(255);
    L.ring_period = dft_visit_period(d);
    L.ring = L.ring_period > 2 ? ar.take<char>((size_t)(L.ring_period - 2) * 3 * Ld * plane * es) : nullptr;
    ar.off = (ar.off + 255) & ~size_t(255);
}

template <class R> class Zone final : public ZoneBase {
public:
    using CR = Cx<R>;
    zda_zone_desc d;
    std::vector<double> omega;
    GridTables g;
    ZoneLayout<R> L;
    cudaStream_t st;
    int max_steps, pitch, cap_terms;
    size_t es, plane, fplane, fvol;
    int Ld, Nrd, F;
    int mk0, mk1;                     // material planes held per voxel: the design layer, or all of them (eps_volume)
    int cur = 0;                      // which field buffer holds the current state
    int kernel_opt = ZDA_KERNEL_AUTO;
    int adj_monitor_dft = 0;
    // experiment / tuning options (zda_set_option): 0 = the plan's own choice
    int opt_tj = 0, opt_chunk = 0, opt_cluster = 0, opt_period = 0, opt_split_graph = 1;
    int check_every = 0;              // ZDA_OPT_CHECK_EVERY: non-finite check of E every K steps of a run (0: off)
    long long launches = 0;
    char* ws_base = nullptr;
    size_t ws_bytes = 0;
    // state flags
    bool have_src[2] = {false, false};
    int n_terms[2] = {0, 0}, tab_len[2] = {0, 0};
    bool have_fwd = false, have_adj = false, have_density = false;
    bool have_focal = false;          // R20 weights held in the adjoint run's monitor accumulators (dft_mon[1])
    double focal_u[ZDA_MAX_FREQ];
    double dens_eps0 = 0, dens_eps_h = 0, dens_sigma = 0, dens_beta = 0, dens_eta = 0;
    double dens_conic_radius = 0;     // > 0: the conic filter (R22) instead of the Gaussian
    std::vector<double> eps_bg;
    std::string kname;
    FusedPlan<R> fused;
    Fused2Plan<R> fused2;

    Zone(const zda_zone_desc& desc, cudaStream_t s, int ms) : d(desc), st(s), max_steps(ms) {
        omega.assign(desc.omega, desc.omega + desc.n_freq);
        d.omega = omega.data();
        build_grid_tables(d, g);
        pitch = g.pitch;
        es = d.complex_fields ? 2 * sizeof(R) : sizeof(R);
        plane = (size_t)pitch * d.Nphi;
        fplane = (size_t)pitch * (d.Nphi + 2 * field_ghost(d));
        fvol = fplane * d.Nz;
        Ld = d.design_k1 - d.design_k0;
        Nrd = d.design_i1 - d.design_i0;
        F = d.n_freq;
        cap_terms = std::max(2, d.complex_fields ? F : 2 * F);
        mk0 = d.eps_volume ? 0 : d.design_k0;
        mk1 = d.eps_volume ? d.Nz : d.design_k1;
    }

    cudaStream_t stream() const override { return st; }
    void workspace_range(const char** lo, const char** hi) const override { *lo = ws_base; *hi = ws_base + ws_bytes; }
    long long launch_count() const override { return launches; }
    const char* kernel_name() const override { return kname.c_str(); }

    int init(const double* eps_bg_z, void* ws, size_t bytes) {
        Arena ar;
        ar.base = (char*)ws;
        carve<R>(d, max_steps, pitch, ar, L);
        if (ar.off > bytes) return fail(ZDA_E_NOMEM, "workspace has %zu bytes, need %zu", bytes, ar.off);
        ws_base = (char*)ws;
        ws_bytes = ar.off;
        // a1: the 1-D tables (rounded once to R).  Every host table is built BEFORE the first upload, so that running out of
        // host memory (std::bad_alloc -> ZDA_E_NOMEM at the ABI) leaves nothing half-initialised on the device.
        std::vector<R> h((size_t)RC_COUNT * pitch, R(0));
        for (int t = 0; t < RC_COUNT; ++t)
            for (int i = 0; i < d.Nr; ++i) h[(size_t)t * pitch + i] = (R)g.rc[t][i];
        for (int i = d.Nr; i < pitch; ++i) h[(size_t)RC_IK_I * pitch + i] = h[(size_t)RC_IK_H * pitch + i] = R(1);
        eps_bg.assign(d.Nz, 1.0);
        if (eps_bg_z) eps_bg.assign(eps_bg_z, eps_bg_z + d.Nz);
        std::vector<R> hz((size_t)ZC_COUNT * d.Nz, R(0));
        for (int t = 0; t < 6; ++t)
            for (int k = 0; k < d.Nz; ++k) hz[(size_t)t * d.Nz + k] = (R)g.zc[t][k];
        for (int k = 0; k < d.Nz; ++k) {
            hz[(size_t)ZC_CE_BG * d.Nz + k] = (R)(d.dt / eps_bg[k]);     // cE = dt / eps, once per voxel
            hz[(size_t)ZC_CE_AXIS * d.Nz + k] = (R)(d.dt / eps_bg[k]);
        }
        // DFT twiddles (R8): dt exp(+i omega_f (n+1) dt), phase evaluated in double exactly as written
        std::vector<CR> tw((size_t)max_steps * F);
        for (int n = 0; n < max_steps; ++n)
            for (int f = 0; f < F; ++f) {
                const double ph = omega[f] * ((double)(n + 1) * d.dt);
                tw[(size_t)n * F + f] = CR{(R)(d.dt * std::cos(ph)), (R)(d.dt * std::sin(ph))};
            }
        ZDA_CUDA_OK(cudaMemcpyAsync(L.rc, h.data(), h.size() * sizeof(R), cudaMemcpyHostToDevice, st));
        ZDA_CUDA_OK(cudaMemcpyAsync(L.zc, hz.data(), hz.size() * sizeof(R), cudaMemcpyHostToDevice, st));
        ZDA_CUDA_OK(cudaMemcpyAsync(L.tw, tw.data(), tw.size() * sizeof(CR), cudaMemcpyHostToDevice, st));
        // the material planes start as background (filled on the device from the 1-D table)
        fill_cE_bg_kernel<R><<<148 * 8, 256, 0, st>>>(L.cE_design, L.zc, d.Nz, mk0, mk1 - mk0, plane);
        ++launches;
        ZDA_CUDA_OK(cudaGetLastError());
        ZDA_CUDA_OK(cudaMemsetAsync(ws_base + L.state_begin, 0, L.state_end - L.state_begin, st));
        for (int w = 0; w < 2; ++w) {
            ZDA_CUDA_OK(cudaMemsetAsync(L.dft_design[w], 0, (size_t)F * 3 * Ld * plane * sizeof(CR), st));
            ZDA_CUDA_OK(cudaMemsetAsync(L.dft_mon[w], 0, (size_t)F * 3 * plane * sizeof(CR), st));
            for (int c = 0; c < 2; ++c) ZDA_CUDA_OK(cudaMemsetAsync(L.A[w][c], 0, (size_t)cap_terms * plane * es, st));
        }
        ZDA_CUDA_OK(cudaStreamSynchronize(st));   // host staging vectors go out of scope
        int rc = select_kernel();
        if (rc != ZDA_OK) return rc;
        return ZDA_OK;
    }

    bool fused_applicable() const {
        return FusedPlan<R>::supported(d);
    }
    bool fused2_applicable() const { return fused_applicable() && Fused2Plan<R>::supported(d) && !d.rpml_exact; }   // R25: one-step kernels only
    bool use_fused2() const {
        return kernel_opt == ZDA_KERNEL_FUSED2 || (kernel_opt == ZDA_KERNEL_AUTO && fused2_applicable() && auto_prefers_fused2());
    }
    bool use_fused() const {
        return kernel_opt == ZDA_KERNEL_FUSED ||
               (kernel_opt == ZDA_KERNEL_AUTO && fused_applicable() && !(fused2_applicable() && auto_prefers_fused2()));
    }
    // the persistent kernel wants the whole state (fields + auxiliaries) to live in L2 (126 MB)
    bool persist_applicable() const { return L.state_end - L.state_begin <= (size_t)96 << 20; }
    bool concurrent_hint = false;     // set by the zone schedulers while zones on other streams are in flight
    bool use_persist() const {
        return kernel_opt == ZDA_KERNEL_PERSIST ||
               (kernel_opt == ZDA_KERNEL_AUTO && !fused_applicable() && persist_applicable() && !concurrent_hint);
    }
    int hint_concurrent(bool on) override {
        if (on == concurrent_hint) return ZDA_OK;
        concurrent_hint = on;
        return select_kernel();
    }
    // Two steps per pass wherever the kernel applies (two ghost rows: Nphi >= 16, no axis, no exact r-PML).  With its lean
    // interior body it measured faster than the one-step kernel on every shape swept (profiles/r02_captures.md, Gvox/s
    // two-step / one-step): config4 117.1 / 91.1, config3 62.5 / 49.8, config2 97.5 / 82.1, 200 x 200 x 160 40.7 / 36.1,
    // 1274 x 32 x 160 54.1 / 43.9 (real) and 39.6 / 36.6 (complex), 1134 x 64 x 160 60.3 / 57.4.  Thin wedges (Nphi < 16) keep
    // the one-step kernel: their layout has one ghost row per side.
    bool auto_prefers_fused2() const { return true; }
    int dft_period_in_use() const {
        const bool f2 = use_fused2(), f1 = use_fused();
        return ((f1 || f2) && L.ring) ? (opt_period ? opt_period : L.ring_period) : 2;
    }
    // Bytes per time step that the schedule in use moves through HBM if every halo re-read hits L2 (bench.py's
    // roofline.schedule_bytes); out = {fields, CPML psi, dt/eps, DFT accumulators + ring, halo re-reads if NONE hit L2}.
    int schedule_bytes(int which, double* out) override {
        const bool f2 = use_fused2(), f1 = use_fused();
        const double V = (double)d.Nr * d.Nphi * d.Nz, esd = (double)es, passes = f2 ? 0.5 : 1.0;
        out[0] = (f1 || f2) ? 12.0 * esd * V * passes : 18.0 * esd * V;     // each field read once + written once per pass;
                                                                             // split: the E pass re-reads H, the H pass E
        const double slab = (double)(d.npml_z_lo + d.npml_z_hi) * d.Nr * d.Nphi + (double)(d.npml_r_lo + d.npml_r_hi) * d.Nphi * d.Nz;
        out[1] = 4.0 * 2.0 * esd * slab * passes;                            // four psi per slab voxel, read + written
        out[2] = (double)sizeof(R) * (mk1 - mk0) * d.Nr * d.Nphi * passes;
        const double acc = 3.0 * F * 2.0 * sizeof(CR);                        // one voxel's accumulators, read + written
        const double mon_every = (f1 || f2) ? 2.0 : 1.0;
        double dft = (which == ZDA_FWD || adj_monitor_dft) ? acc * d.Nr * d.Nphi / mon_every : 0.0;
        const double Vd = (double)Nrd * d.Nphi * Ld;
        const int p = dft_period_in_use();
        if (!(f1 || f2)) dft += acc * Vd;
        else if (p == 2) dft += (acc + (f2 ? 0.0 : 3.0 * esd)) / 2.0 * Vd;   // one-step kernel: re-reads E^n every second launch
        else dft += (acc + 3.0 * esd * (2 * p - 2)) / p * Vd;                // p - 2 ring stores + p reads of E per group
        out[3] = dft;
        double halo = 0.0;
        if (f1) halo = 6.0 * esd * V * ((fused.tj + 2.0) / fused.tj * 34.0 / 32.0 - 1.0);
        if (f2) {
            const int vec = (int)(16 / es), lo = (2 + vec - 1) / vec;
            halo = 6.0 * esd * V * 0.5 * ((fused2.tj + 4.0) / fused2.tj * 33.0 / (31.0 - lo) * (fused2.G.chunk + 3.0) / fused2.G.chunk - 1.0);
        }
        out[4] = halo;
        return ZDA_OK;
    }
    int select_kernel() {
        if ((kernel_opt == ZDA_KERNEL_FUSED || kernel_opt == ZDA_KERNEL_FUSED2) && !fused_applicable())
            return fail(ZDA_E_BADARG, "fused kernel does not apply to this zone (axis zone or unsupported shape)");
        if (kernel_opt == ZDA_KERNEL_FUSED2 && !fused2_applicable())
            return fail(ZDA_E_BADARG, "the two-step kernel needs Nphi >= 16 (a field layout with two ghost rows) and no exact outer r-PML; use ZDA_KERNEL_FUSED");
        if (kernel_opt == ZDA_KERNEL_PERSIST && !persist_applicable())
            return fail(ZDA_E_BADARG, "the persistent kernel needs the zone's state (%zu MB) to fit 96 MB", (L.state_end - L.state_begin) >> 20);
        if (use_persist()) {
            int rc = prepare_persist();
            if (rc != ZDA_OK) return rc;
            return ZDA_OK;
        }
        if (use_fused2()) {
            int rc = fused2.prepare(d, pitch, L.fbase, L.fstride, opt_tj, opt_chunk, opt_cluster);
            if (rc != ZDA_OK) return rc;
            kname = std::string(fused2.name()) + ", dft visit period " + std::to_string(dft_period_in_use());
            return ZDA_OK;
        }
        if (use_fused()) {
            int rc = fused.prepare(d, pitch, L.fbase, L.fstride, opt_tj, opt_chunk, opt_cluster);
            if (rc != ZDA_OK) return rc;
            kname = std::string(fused.name()) + ", dft visit period " + std::to_string(dft_period_in_use());
            return ZDA_OK;
        }
        kname = "split";
        return ZDA_OK;
    }

    int set_option(int option, int value) override {
        if (option == ZDA_OPT_KERNEL) {
            if (value < ZDA_KERNEL_AUTO || value > ZDA_KERNEL_PERSIST) return fail(ZDA_E_BADARG, "bad kernel option");
            const int old = kernel_opt;
            kernel_opt = value;
            int rc = select_kernel();
            if (rc != ZDA_OK) { kernel_opt = old; select_kernel(); }
            return rc;
        }
        auto replan = [&](int& slot, int v) {
            const int old = slot;
            slot = v;
            int rc = select_kernel();
            if (rc != ZDA_OK) { slot = old; select_kernel(); }
            return rc;
        };
        if (option == ZDA_OPT_FUSED_TJ) {
            if (value != 0 && value != 5 && value != 6 && value != 7 && value != 9 && value != 13)
                return fail(ZDA_E_BADARG, "ZDA_OPT_FUSED_TJ: 0 (auto), 6 or 7 (one-step kernel), 5, 9 or 13 (two-step kernel)");
            return replan(opt_tj, value);
        }
        if (option == ZDA_OPT_FUSED_CHUNK) {
            if (value < 0) return fail(ZDA_E_BADARG, "ZDA_OPT_FUSED_CHUNK: 0 (auto) or a number of planes");
            return replan(opt_chunk, value);
        }
        if (option == ZDA_OPT_FUSED_CLUSTER) {
            if (value < 0 || value > 8) return fail(ZDA_E_BADARG, "ZDA_OPT_FUSED_CLUSTER: 0 (auto) or 1..8");
            return replan(opt_cluster, value);
        }
        if (option == ZDA_OPT_DFT_PERIOD) {
            if (value != 0 && value != 2 && value != 4 && value != 8) return fail(ZDA_E_BADARG, "ZDA_OPT_DFT_PERIOD: 0 (auto), 2, 4 or 8");
            if (value > std::max(2, L.ring_period))
                return fail(ZDA_E_BADARG, "ZDA_OPT_DFT_PERIOD %d exceeds the ring this zone's workspace holds (period %d)", value, L.ring_period);
            opt_period = value;
            return select_kernel();
        }
        if (option == ZDA_OPT_SPLIT_GRAPH) { opt_split_graph = value ? 1 : 0; return ZDA_OK; }
        if (option == ZDA_OPT_CHECK_EVERY) {
            if (value < 0) return fail(ZDA_E_BADARG, "ZDA_OPT_CHECK_EVERY: K >= 0");
            check_every = value;
            return ZDA_OK;
        }
        if (option == ZDA_OPT_ADJ_MONITOR_DFT) {
            if (value && have_focal)
                return fail(ZDA_E_STATE, "the adjoint monitor DFT shares its buffer with the focal weights (zda_set_focal_weights)");
            adj_monitor_dft = value ? 1 : 0;
            return ZDA_OK;
        }
        return fail(ZDA_E_BADARG, "unknown option %d", option);
    }

    // ---- materials -------------------------------------------------------------------------
    int refresh_axis_cE() {
        if (!d.has_axis) return ZDA_OK;
        axis_cE_kernel<R><<<(d.Nz + 127) / 128, 128, 0, st>>>(L.cE_design, L.zc, L.zc + (size_t)ZC_CE_AXIS * d.Nz, d.Nz,
                                                              d.Nphi, pitch, mk0, mk1, (R)d.dt);
        ++launches;
        ZDA_CUDA_OK(cudaGetLastError());
        return ZDA_OK;
    }

    // dt/eps of the design layer inside the material planes
    R* cE_layer() const { return L.cE_design + (size_t)(d.design_k0 - mk0) * plane; }

    // per-voxel eps over the whole zone (north_star "per-voxel eps"; SURVEY 8(b) `eps /*Nr*Nphi*Nz*/`), dense [k][j][i];
    // streamed through the design-box staging buffer a few planes at a time when it comes from the host
    int set_eps_volume(const void* eps, int on_host) override {
        if (!d.eps_volume) return fail(ZDA_E_STATE, "zda_set_eps_volume needs desc.eps_volume = 1 at zone creation");
        const size_t rows_total = (size_t)d.Nz * d.Nphi;
        const R* src = (const R*)eps;
        const size_t cap_rows = std::max<size_t>(1, ((size_t)Nrd * d.Nphi * Ld) / d.Nr);   // rows the staging buffer holds
        for (size_t r0 = 0; r0 < rows_total;) {
            const size_t rows = on_host ? std::min(cap_rows, rows_total - r0) : rows_total;
            const R* chunk = src + r0 * d.Nr;
            if (on_host) {
                ZDA_CUDA_OK(cudaMemcpyAsync(L.staging, chunk, rows * d.Nr * sizeof(R), cudaMemcpyHostToDevice, st));
                chunk = L.staging;
            }
            const int blocks = (int)std::min<size_t>((rows * d.Nr + 255) / 256, 148 * 16);
            eps_volume_to_cE_kernel<R><<<blocks, 256, 0, st>>>(chunk, L.cE_design + r0 * pitch, d.Nr, rows, pitch, (R)d.dt);
            ++launches;
            ZDA_CUDA_OK(cudaGetLastError());
            if (on_host) ZDA_CUDA_OK(cudaStreamSynchronize(st));   // the staging buffer is reused by the next chunk
            r0 += rows;
        }
        have_density = false;
        return refresh_axis_cE();
    }

    int set_design_eps(const void* eps, int on_host) override {
        const size_t n = (size_t)Nrd * d.Nphi * Ld;
        const R* src = (const R*)eps;
        if (on_host) {
            ZDA_CUDA_OK(cudaMemcpyAsync(L.staging, eps, n * sizeof(R), cudaMemcpyHostToDevice, st));
            src = L.staging;
        }
        const int blocks = (int)std::min<size_t>((n + 255) / 256, 148 * 16);
        eps_to_cE_kernel<R><<<blocks, 256, 0, st>>>(src, cE_layer(), Nrd, d.Nphi, Ld, pitch, d.design_i0, (R)d.dt);
        ++launches;
        ZDA_CUDA_OK(cudaGetLastError());
        have_density = false;
        int rc = refresh_axis_cE();
        if (rc != ZDA_OK) return rc;
        if (on_host) ZDA_CUDA_OK(cudaStreamSynchronize(st));
        return ZDA_OK;
    }

    FilterW<R> filter_weights(double sigma) const {
        FilterW<R> W;
        W.Rad = (int)std::ceil(3.0 * sigma);
        double sum = 0.0;
        std::vector<double> w(2 * W.Rad + 1);
        for (int t = -W.Rad; t <= W.Rad; ++t) { w[t + W.Rad] = std::exp(-0.5 * (t / sigma) * (t / sigma)); sum += w[t + W.Rad]; }
        for (int t = 0; t <= 2 * W.Rad; ++t) W.w[t] = (R)(w[t] / sum);
        return W;
    }

    ConicP<R> conic_params(double radius) const {
        ConicP<R> C;
        const double r_first = d.r_in + (d.design_i0 + 0.5) * d.dr;
        C.r_first = (R)r_first; C.dr = (R)d.dr; C.dphi = (R)d.dphi; C.inv_R = (R)(1.0 / radius);
        C.a_max = std::min((int)std::floor(radius / d.dr), Nrd - 1);
        C.b_max = (int)std::floor(radius / (r_first * d.dphi));
        return C;
    }

    // filter_mode 0: separable Gaussian, width = sigma in cells (R13); 1: conic, width = radius in length units (R22)
    int set_density(const void* rho, int on_host, int filter_mode, double eps0, double eps_h, double width, double beta,
                    double eta) override {
        const size_t n2 = (size_t)Nrd * d.Nphi;
        const dim3 grid((Nrd + 127) / 128, d.Nphi);
        if (filter_mode == 1) {
            const ConicP<R> C = conic_params(width);
            if (C.b_max > 4096) return fail(ZDA_E_BADARG, "conic filter reaches %d phi cells at the inner design radius", C.b_max);
            ZDA_CUDA_OK(cudaMemcpyAsync(L.rho, rho, n2 * sizeof(R), on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, st));
            conic_kernel<R, 0><<<grid, 128, 0, st>>>(L.rho, L.rho_f, Nrd, d.Nphi, C);
            launches += 1;
        } else {
            ZDA_CUDA_OK(cudaMemcpyAsync(L.rho, rho, n2 * sizeof(R), on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, st));
            const FilterW<R> W = filter_weights(width);
            filter_r_kernel<R><<<grid, 128, 0, st>>>(L.rho, L.tmp2d, Nrd, d.Nphi, W);
            filter_phi_kernel<R><<<grid, 128, 0, st>>>(L.tmp2d, L.rho_f, Nrd, d.Nphi, W);
            launches += 2;
        }
        project_extrude_kernel<R><<<grid, 128, 0, st>>>(L.rho_f, cE_layer(), Nrd, d.Nphi, Ld, pitch, d.design_i0,
                                                        (R)d.dt, (R)eps0, (R)eps_h, (R)beta, (R)eta);
        launches += 1;
        ZDA_CUDA_OK(cudaGetLastError());
        dens_eps0 = eps0; dens_eps_h = eps_h; dens_beta = beta; dens_eta = eta;
        dens_sigma = filter_mode == 1 ? 0.0 : width;
        dens_conic_radius = filter_mode == 1 ? width : 0.0;
        have_density = true;
        int rc = refresh_axis_cE();
        if (rc != ZDA_OK) return rc;
        if (on_host) ZDA_CUDA_OK(cudaStreamSynchronize(st));
        return ZDA_OK;
    }

    // ---- sources ---------------------------------------------------------------------------
    int upload_sheet(int which, int nt, const void* A_r, const void* A_phi, int on_host) {
        // dense [q][j][Nr] -> pitched [q][j][pitch]
        const cudaMemcpyKind kind = on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
        const void* src[2] = {A_r, A_phi};
        for (int c = 0; c < 2; ++c)
            ZDA_CUDA_OK(cudaMemcpy2DAsync(L.A[which][c], (size_t)pitch * es, src[c], (size_t)d.Nr * es, (size_t)d.Nr * es,
                                          (size_t)nt * d.Nphi, kind, st));
        return ZDA_OK;
    }
    int upload_table(int which, int nt, const double* tab_re_im, int Nt) {
        // host doubles (interleaved re, im when complex) -> device field elements
        if (Nt > max_steps) return fail(ZDA_E_BADARG, "table length %d exceeds max_steps %d", Nt, max_steps);
        const int comps = d.complex_fields ? 2 : 1;
        std::vector<R> h((size_t)nt * Nt * comps);
        for (size_t t = 0; t < h.size(); ++t) h[t] = (R)tab_re_im[t];
        ZDA_CUDA_OK(cudaMemcpyAsync(L.s_tab[which], h.data(), h.size() * sizeof(R), cudaMemcpyHostToDevice, st));
        ZDA_CUDA_OK(cudaStreamSynchronize(st));
        n_terms[which] = nt;
        tab_len[which] = Nt;
        have_src[which] = true;
        return ZDA_OK;
    }
    int set_source(int nt, const void* A_r, const void* A_phi, int on_host, const double* s_table, int Nt) override {
        if (nt > cap_terms) return fail(ZDA_E_BADARG, "n_terms %d exceeds the zone's capacity %d", nt, cap_terms);
        int rc = upload_sheet(0, nt, A_r, A_phi, on_host);
        if (rc != ZDA_OK) return rc;
        return upload_table(0, nt, s_table, Nt);
    }

    // ---- time loop -------------------------------------------------------------------------
    template <class T> void fill_params(StepParams<T>& P, int which) {
        P.Nr = d.Nr; P.Nphi = d.Nphi; P.Nz = d.Nz; P.pitch = pitch; P.fplane = fplane; P.ghost = field_ghost(d);
        P.has_axis = d.has_axis;
        P.p_is_one = (d.phase_re == 1.0 && d.phase_im == 0.0);
        P.dt = (R)d.dt; P.inv_dr = (R)(1.0 / d.dr); P.inv_dz = (R)(1.0 / d.dz);
        P.pr = (R)d.phase_re;
        P.pi = (R)(which == ZDA_ADJ ? -d.phase_im : d.phase_im);   // R12: the adjoint run carries the conjugate phase
        P.rc = L.rc; P.zc = L.zc;
        P.rpml_exact = d.rpml_exact;
        P.npr_lo = d.npml_r_lo; P.npr_hi = d.npml_r_hi; P.npz_lo = d.npml_z_lo; P.npz_hi = d.npml_z_hi;
        P.cE_design = L.cE_design;
        P.mk0 = mk0; P.mk1 = mk1;
        P.di0 = d.design_i0; P.di1 = d.design_i1; P.dk0 = d.design_k0; P.dk1 = d.design_k1;
        P.axis_mean = (const T*)L.axis_mean;
        P.A_r = (const T*)L.A[which][0]; P.A_phi = (const T*)L.A[which][1];
        P.s_tab = (const T*)L.s_tab[which];
        P.n_terms = have_src[which] ? n_terms[which] : 0;
        P.tab_len = tab_len[which];
        P.src_k = which == ZDA_ADJ ? d.monitor_k : d.source_k;
        P.F = F; P.tw = L.tw;
        P.dft_design = L.dft_design[which];
        P.dft_mon = (which == ZDA_FWD || adj_monitor_dft) ? L.dft_mon[which] : nullptr;
        P.mon_k = P.dft_mon ? d.monitor_k : -1;
        P.n = 0;
        P.n_dev = nullptr;
        P.ring_store = nullptr;
        P.ring_store_b = nullptr;
    }
    // ZDA_OPT_CHECK_EVERY (SURVEY 5 "NaN/Inf check every K steps, error code through the C ABI"): after step n of a run,
    // every K-th step, scan E for non-finite values; synchronises and stops the run with ZDA_E_NAN when there are any.
    template <class T> int periodic_check(int n) {
        if (check_every <= 0 || (n + 1) % check_every != 0) return ZDA_OK;
        int* flag = L.step_counter + 16;
        ZDA_CUDA_OK(cudaMemsetAsync(flag, 0, sizeof(int), st));
        for (int c = 0; c < 3; ++c) nonfinite_flag_kernel<T><<<148 * 8, 256, 0, st>>>((const T*)L.E[cur][c], fvol, flag);
        launches += 3;
        ZDA_CUDA_OK(cudaGetLastError());
        int h = 0;
        ZDA_CUDA_OK(cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, st));
        ZDA_CUDA_OK(cudaStreamSynchronize(st));
        if (h) return fail(ZDA_E_NAN, "non-finite E after step %d of the run (checked every %d steps)", n + 1, check_every);
        return ZDA_OK;
    }
    // in_place: the split kernels update the current buffers; the fused kernels read `cur` and write the other one
    template <class T> void bind_buffers(StepParams<T>& P, bool in_place = false) {
        const int o = in_place ? cur : (cur ^ 1);
        for (int c = 0; c < 2; ++c) {
            P.psiE_z[c] = (T*)L.psiE_z[cur][c]; P.psiE_r[c] = (T*)L.psiE_r[cur][c];
            P.psiE_z_out[c] = (T*)L.psiE_z[o][c]; P.psiE_r_out[c] = (T*)L.psiE_r[o][c];
            P.chiH[c] = (T*)L.chiH[cur][c]; P.chiH_out[c] = (T*)L.chiH[o][c];
            P.chiE[c] = (T*)L.chiE[cur][c]; P.chiE_out[c] = (T*)L.chiE[o][c];
        }
        for (int c = 0; c < 3; ++c) {
            P.E[c] = (T*)L.E[cur][c]; P.H[c] = (T*)L.H[cur][c];
            P.Eout[c] = (T*)L.E[cur ^ 1][c]; P.Hout[c] = (T*)L.H[cur ^ 1][c];
        }
        for (int c = 0; c < 2; ++c) {
            P.psiH_z[c] = (T*)L.psiH_z[cur][c]; P.psiH_r[c] = (T*)L.psiH_r[cur][c];
            P.psiH_z_out[c] = (T*)L.psiH_z[cur ^ 1][c]; P.psiH_r_out[c] = (T*)L.psiH_r[cur ^ 1][c];
        }
    }

    // reset: all fields, CPML auxiliaries and this run's accumulators; fills the launch-invariant parameters
    template <class T> int begin_run(StepParams<T>& P, int which, int n_steps) {
        if (n_steps > max_steps) return fail(ZDA_E_BADARG, "n_steps %d exceeds max_steps %d", n_steps, max_steps);
        // Only time buffer 0 starts a run: the first pass reads it and overwrites every cell of buffer 1 that is ever read
        // (zone creation zeroed both once, so the row padding stays finite).  Half the memset of round 1 (24 GB on config4).
        {
            const int npz = d.npml_z_lo + d.npml_z_hi, npr = d.npml_r_lo + d.npml_r_hi;
            const size_t zsz = (size_t)std::max(npz, 1) * plane * es, rsz = (size_t)d.Nz * d.Nphi * std::max(npr, 1) * es;
            ZDA_CUDA_OK(cudaMemsetAsync(L.fbase, 0, 6 * L.fstride, st));
            for (int c = 0; c < 2; ++c) {
                ZDA_CUDA_OK(cudaMemsetAsync(L.psiH_z[0][c], 0, zsz, st));
                ZDA_CUDA_OK(cudaMemsetAsync(L.psiE_z[0][c], 0, zsz, st));
                ZDA_CUDA_OK(cudaMemsetAsync(L.psiH_r[0][c], 0, rsz, st));
                ZDA_CUDA_OK(cudaMemsetAsync(L.psiE_r[0][c], 0, rsz, st));
                if (d.rpml_exact) {
                    ZDA_CUDA_OK(cudaMemsetAsync(L.chiH[0][c], 0, rsz, st));
                    ZDA_CUDA_OK(cudaMemsetAsync(L.chiE[0][c], 0, rsz, st));
                }
            }
            ZDA_CUDA_OK(cudaMemsetAsync(L.axis_mean, 0, (size_t)d.Nz * es, st));
        }
        ZDA_CUDA_OK(cudaMemsetAsync(L.dft_design[which], 0, (size_t)F * 3 * Ld * plane * sizeof(CR), st));
        if (!(which == ZDA_ADJ && have_focal))   // the adjoint run's monitor buffer holds the focal weights (R20)
            ZDA_CUDA_OK(cudaMemsetAsync(L.dft_mon[which], 0, (size_t)F * 3 * plane * sizeof(CR), st));
        cur = 0;
        std::memset(&P, 0, sizeof(P));     // padding too: the split path compares parameter blocks byte-wise
        fill_params(P, which);
        return ZDA_OK;
    }
    // One-step fused kernel, step n of a run: what this launch does with the accumulators and the ring, and its buffers.
    template <class T> void fused_step_setup(StepParams<T>& P, int which, int n, int n_steps, int period) {
        const bool ext = period > 2;          // design-box accumulators visited by dft_visit_kernel every `period` steps
        P.n = n;
        P.dft_design = ext ? nullptr : L.dft_design[which];
        // the fused kernel visits the accumulators it is given (the monitor plane's; the design box's unless `ext`)
        // every second step, and on an odd last step
        P.dft_mode = (n & 1) ? 2 : (n == n_steps - 1 ? 1 : 0);
        const int g0 = n / period * period, g1 = std::min(g0 + period, n_steps), m = g1 - g0, t = n - g0;
        // E^{n+1} is still in a time buffer at the visit (after launch g1 - 1) only for the group's last two steps
        P.ring_store = (ext && t <= m - 3) ? (T*)L.ring + (size_t)t * 3 * Ld * plane : nullptr;
        bind_buffers(P);
    }
    // after the launch of step n: swap the time buffers; the accumulator visit when a group is complete
    template <class T> void fused_step_finish(int which, int n, int n_steps, int period) {
        ++launches;
        cur ^= 1;
        const int g0 = n / period * period, g1 = std::min(g0 + period, n_steps), m = g1 - g0;
        if (period <= 2 || n != g1 - 1) return;
        const size_t slot_elems = (size_t)3 * Ld * plane;
        VisitParams<T> V;
        V.m = m; V.F = F; V.n0 = g0; V.Nphi = d.Nphi; V.Ld = Ld; V.pitch = pitch;
        V.di0 = d.design_i0; V.di1 = d.design_i1; V.plane = plane;
        V.dft = L.dft_design[which]; V.tw = L.tw;
        for (int q = 0; q < m; ++q) {
            if (q <= m - 3) {          // ring slot q
                for (int c = 0; c < 3; ++c) V.src[q].p[c] = (const T*)L.ring + (size_t)q * slot_elems + (size_t)c * Ld * plane;
                V.src[q].kstride = plane;
            } else {                    // time buffer: E^{g1} is in `cur` now, E^{g1-1} in the other one
                const int b = (q == m - 1) ? cur : (cur ^ 1);
                for (int c = 0; c < 3; ++c)
                    V.src[q].p[c] = (const T*)L.E[b][c] + (size_t)d.design_k0 * fplane + (size_t)field_ghost(d) * pitch;   // storage row j + FIELD_GHOST
                V.src[q].kstride = fplane;
            }
        }
        const int vec = (int)(16 / es);
        const int groups = (d.design_i1 + vec - 1) / vec - d.design_i0 / vec;
        dft_visit_kernel<T><<<dim3((groups + 127) / 128, d.Nphi, Ld), 128, 0, st>>>(V);
        ++launches;
    }
    int fused_period() const { return L.ring ? (opt_period ? opt_period : L.ring_period) : 2; }

    template <class T> int run_T(int which, int n_steps) {
        StepParams<T> P;
        int rc = begin_run(P, which, n_steps);
        if (rc != ZDA_OK) return rc;
        if (use_persist()) return run_persist<T>(P, which, n_steps);
        if (use_fused2()) return run_fused2<T>(P, which, n_steps);
        if (!use_fused()) {
            const dim3 blk(SPLIT_BX, SPLIT_BY, SPLIT_BZ);
            const dim3 grd((d.Nr + SPLIT_BX - 1) / SPLIT_BX, (d.Nphi + SPLIT_BY - 1) / SPLIT_BY, (d.Nz + SPLIT_BZ - 1) / SPLIT_BZ);
            rc = run_split<T>(P, which, n_steps, grd, blk);
            if (rc != ZDA_OK) return rc;
            ZDA_CUDA_OK(cudaGetLastError());
            return ZDA_OK;
        }
        const int period = fused_period();
        for (int n = 0; n < n_steps; ++n) {
            fused_step_setup(P, which, n, n_steps, period);
            rc = fused.template launch<T>(P, cur, st);
            if (rc != ZDA_OK) return rc;
            fused_step_finish<T>(which, n, n_steps, period);
            rc = periodic_check<T>(n);
            if (rc != ZDA_OK) return rc;
        }
        ZDA_CUDA_OK(cudaGetLastError());
        return ZDA_OK;
    }

    // NEXT-4: this zone and `o` (same shape, same one-step launch plan, same stream) advance together, one launch per time
    // step for both (fused_step_batch_kernel); resets, accumulator visits and results are each zone's own.
    template <class T> int run_batch_T(Zone<R>& o, int which, int n_steps) {
        StepParams<T> P0, P1;
        int rc = begin_run(P0, which, n_steps);
        if (rc == ZDA_OK) rc = o.begin_run(P1, which, n_steps);
        if (rc != ZDA_OK) return rc;
        const int period = fused_period();
        for (int n = 0; n < n_steps; ++n) {
            fused_step_setup(P0, which, n, n_steps, period);
            o.fused_step_setup(P1, which, n, n_steps, period);
            rc = fused.template launch_batch<T>(P0, P1, o.fused, cur, st);
            if (rc != ZDA_OK) return rc;
            fused_step_finish<T>(which, n, n_steps, period);
            o.template fused_step_finish<T>(which, n, n_steps, period);
            --o.launches;               // the step was ONE launch for both
        }
        ZDA_CUDA_OK(cudaGetLastError());
        return ZDA_OK;
    }
    // why (or whether) two zones can share their launches: nullptr = they can
    const char* batch_obstacle(const Zone<R>& o) const {
        if (!use_fused() || !o.use_fused()) return "both zones must run the one-step fused kernel";
        if (st != o.st) return "the zones are on different streams";
        if (d.Nr != o.d.Nr || d.Nphi != o.d.Nphi || d.Nz != o.d.Nz || d.complex_fields != o.d.complex_fields ||
            d.npml_r_lo != o.d.npml_r_lo || d.npml_r_hi != o.d.npml_r_hi || d.npml_z_lo != o.d.npml_z_lo ||
            d.npml_z_hi != o.d.npml_z_hi || d.n_freq != o.d.n_freq || d.design_i0 != o.d.design_i0 ||
            d.design_i1 != o.d.design_i1 || d.design_k0 != o.d.design_k0 || d.design_k1 != o.d.design_k1 ||
            d.eps_volume != o.d.eps_volume)
            return "the zones differ in grid, CPML, design box or number of frequencies";
        if (fused.tj != o.fused.tj || fused.G.chunk != o.fused.G.chunk || fused.G.cluster != o.fused.G.cluster ||
            fused_period() != o.fused_period())
            return "the zones have different launch plans";
        if (check_every || o.check_every) return "ZDA_OPT_CHECK_EVERY is set";
        if (d.rpml_exact || o.d.rpml_exact) return "the exact outer r-PML (rpml_exact) has no batched kernel";
        return nullptr;
    }
    bool can_batch_with(ZoneBase* other) const override {
        const Zone<R>* o = dynamic_cast<const Zone<R>*>(other);
        return o && o != this && batch_obstacle(*o) == nullptr;
    }
    int run_batch(ZoneBase* other, int which, int n_steps) override {
        Zone<R>* o = dynamic_cast<Zone<R>*>(other);
        if (!o || o == this) return fail(ZDA_E_BADARG, "the two zones must be distinct and of one precision");
        if (const char* why = batch_obstacle(*o)) return fail(ZDA_E_BADARG, "zones cannot share a launch: %s", why);
        if (which == ZDA_ADJ && (!have_src[1] || !o->have_src[1]))
            return fail(ZDA_E_STATE, "a batched adjoint run needs zda_build_adjoint_source on both zones");
        int rc = d.complex_fields ? run_batch_T<CR>(*o, which, n_steps) : run_batch_T<R>(*o, which, n_steps);
        if (rc != ZDA_OK) return rc;
        for (Zone<R>* z : {this, o}) {
            if (which == ZDA_FWD) { z->have_fwd = true; z->have_adj = false; z->have_src[1] = false; }
            else z->have_adj = true;
        }
        return ZDA_OK;
    }

    // Small zones: one cooperative launch steps the whole run (persist_kernel); with ZDA_OPT_CHECK_EVERY one launch per K steps.
    int persist_blocks = 0;
    int prepare_persist() {
        int dev = 0, sms = 148, per_sm_r = 0, per_sm_c = 0, coop = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        if (!coop) return fail(ZDA_E_CUDA, "this device does not support cooperative launches");
        ZDA_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_r, persist_kernel<R>, PERSIST_THREADS, 0));
        ZDA_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_c, persist_kernel<CR>, PERSIST_THREADS, 0));
        const int per_sm = std::max(1, std::min(d.complex_fields ? per_sm_c : per_sm_r, opt_chunk > 0 ? opt_chunk : 1));
        const long want = ((long)d.Nr * d.Nphi * d.Nz + PERSIST_THREADS - 1) / PERSIST_THREADS;
        persist_blocks = (int)std::max<long>(1, std::min<long>((long)sms * per_sm, want));
        char buf[160];
        snprintf(buf, sizeof(buf), "persist(one cooperative launch per run, %d x 512 thr, grid barrier between the H and E passes, state %zu MB in L2)",
                 persist_blocks, (L.state_end - L.state_begin) >> 20);
        kname = buf;
        return ZDA_OK;
    }
    template <class T> int run_persist(StepParams<T>& P, int which, int n_steps) {
        (void)which;
        P.dft_mode = 1;
        P.n_dev = nullptr;
        bind_buffers(P, true);
        const int seg = check_every > 0 ? check_every : n_steps;
        for (int n0 = 0; n0 < n_steps; n0 += seg) {
            int ns = std::min(seg, n_steps - n0), n0v = n0;
            void* args[] = {(void*)&P, (void*)&n0v, (void*)&ns};
            ZDA_CUDA_OK(cudaLaunchCooperativeKernel((const void*)persist_kernel<T>, dim3(persist_blocks), dim3(PERSIST_THREADS), args, 0, st));
            ++launches;
            int rc = periodic_check<T>(n0 + ns - 1);
            if (rc != ZDA_OK) return rc;
        }
        ZDA_CUDA_OK(cudaGetLastError());
        return ZDA_OK;
    }
    // Two steps per launch (zda_kernels_fused2.cuh).  An odd last step is made by the split kernels (in place on the
    // current buffers; their own every-step DFT adds the last term, after every earlier one).
    template <class T> int run_fused2(StepParams<T>& P, int which, int n_steps) {
        const int n_pairs = n_steps / 2;
        const int period = L.ring ? (opt_period ? opt_period : L.ring_period) : 2;
        const bool ext = period > 2;
        const size_t slot_elems = (size_t)3 * Ld * plane;
        auto ring_slot = [&](int s) { return (T*)L.ring + (size_t)s * slot_elems; };
        for (int l = 0; l < n_pairs; ++l) {
            const int n = 2 * l;
            P.n = n;
            P.dft_mode = 2;
            const int g0 = n / period * period, g1 = std::min(g0 + period, 2 * n_pairs), nl = (g1 - g0) / 2, lg = (n - g0) / 2;
            P.dft_design = ext ? nullptr : L.dft_design[which];
            P.ring_store = ext ? ring_slot(lg) : nullptr;
            P.ring_store_b = (ext && lg <= nl - 3) ? ring_slot(period / 2 + lg) : nullptr;
            bind_buffers(P);
            int rc = fused2.template launch<T>(P, cur, st);
            if (rc != ZDA_OK) return rc;
            ++launches;
            cur ^= 1;
            if (ext && lg == nl - 1) {
                VisitParams<T> V;
                const int m = g1 - g0;
                V.m = m; V.F = F; V.n0 = g0; V.Nphi = d.Nphi; V.Ld = Ld; V.pitch = pitch;
                V.di0 = d.design_i0; V.di1 = d.design_i1; V.plane = plane;
                V.dft = L.dft_design[which]; V.tw = L.tw;
                for (int q = 0; q < m; ++q) {
                    const int lq = q / 2;
                    const bool in_buffer = (q & 1) && lq >= nl - 2;     // E^{n+2} of the group's last two launches
                    if (!in_buffer) {
                        const T* base = ring_slot((q & 1) ? period / 2 + lq : lq);
                        for (int c = 0; c < 3; ++c) V.src[q].p[c] = base + (size_t)c * Ld * plane;
                        V.src[q].kstride = plane;
                    } else {
                        const int b = (lq == nl - 1) ? cur : (cur ^ 1);
                        for (int c = 0; c < 3; ++c)
                            V.src[q].p[c] = (const T*)L.E[b][c] + (size_t)d.design_k0 * fplane + (size_t)field_ghost(d) * pitch;
                        V.src[q].kstride = fplane;
                    }
                }
                const int vec = (int)(16 / es);
                const int groups = (d.design_i1 + vec - 1) / vec - d.design_i0 / vec;
                dft_visit_kernel<T><<<dim3((groups + 127) / 128, d.Nphi, Ld), 128, 0, st>>>(V);
                ++launches;
            }
            if (check_every > 0 && (n + 2) / check_every > n / check_every) {
                rc = periodic_check<T>((n + 2) / check_every * check_every - 1);
                if (rc != ZDA_OK) return rc;
            }
        }
        if (n_steps & 1) {
            P.n = n_steps - 1;
            P.dft_mode = 1;
            P.dft_design = L.dft_design[which];
            P.ring_store = P.ring_store_b = nullptr;
            P.n_dev = nullptr;
            bind_buffers(P, true);
            const dim3 blk(SPLIT_BX, SPLIT_BY, SPLIT_BZ);
            const dim3 grd((d.Nr + SPLIT_BX - 1) / SPLIT_BX, (d.Nphi + SPLIT_BY - 1) / SPLIT_BY, (d.Nz + SPLIT_BZ - 1) / SPLIT_BZ);
            launch_split_step<T>(P, grd, blk, st);
            launches += d.has_axis ? 3 : 2;
            int rc = periodic_check<T>(n_steps - 1);
            if (rc != ZDA_OK) return rc;
        }
        ZDA_CUDA_OK(cudaGetLastError());
        return ZDA_OK;
    }
    // Split path: the kernels update in place, so with the step index on the device (StepParams::n_dev) every step has
    // the SAME launch parameters: SPLIT_GRAPH_STEPS steps are captured once into a CUDA graph (on a private capture
    // stream: the zone's stream may be the legacy default stream, which cannot capture) and replayed.  Small zones (the
    // one-phi-cell first zone: 2e5 voxels, 3 launches per step) are launch-bound otherwise.
    static constexpr int SPLIT_GRAPH_STEPS = 32;
    cudaStream_t cap_st = nullptr;
    cudaGraphExec_t split_exec[2] = {nullptr, nullptr};
    std::vector<char> split_key[2];
    template <class T> void launch_split_step(const StepParams<T>& P, dim3 grd, dim3 blk, cudaStream_t s) {
        h_update_kernel<T><<<grd, blk, 0, s>>>(P);
        if (d.has_axis) axis_mean_kernel<T><<<(d.Nz + 127) / 128, 128, 0, s>>>(P, (T*)L.axis_mean);
        e_update_kernel<T><<<grd, blk, 0, s>>>(P);
    }
    template <class T> int run_split(StepParams<T>& P, int which, int n_steps, dim3 grd, dim3 blk) {
        const int per_step = d.has_axis ? 3 : 2;
        P.dft_mode = 1;
        bind_buffers(P, true);
        const bool use_graph = n_steps >= 2 * SPLIT_GRAPH_STEPS && opt_split_graph != 0 && check_every == 0;
        int done = 0;
        if (use_graph) {
            P.n = 0;
            P.n_dev = L.step_counter;
            ZDA_CUDA_OK(cudaMemsetAsync(L.step_counter, 0xFF, sizeof(int), st));     // -1: the first H-update makes it 0
            const char* key = reinterpret_cast<const char*>(&P);
            if (!split_exec[which] || split_key[which].size() != sizeof(P) ||
                std::memcmp(split_key[which].data(), key, sizeof(P)) != 0) {
                if (split_exec[which]) { cudaGraphExecDestroy(split_exec[which]); split_exec[which] = nullptr; }
                if (!cap_st) ZDA_CUDA_OK(cudaStreamCreateWithFlags(&cap_st, cudaStreamNonBlocking));
                cudaGraph_t graph = nullptr;
                ZDA_CUDA_OK(cudaStreamBeginCapture(cap_st, cudaStreamCaptureModeThreadLocal));
                for (int n = 0; n < SPLIT_GRAPH_STEPS; ++n) launch_split_step<T>(P, grd, blk, cap_st);
                ZDA_CUDA_OK(cudaStreamEndCapture(cap_st, &graph));
                cudaError_t e = cudaGraphInstantiate(&split_exec[which], graph, 0);
                cudaGraphDestroy(graph);
                if (e != cudaSuccess) return fail(ZDA_E_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
                split_key[which].assign(key, key + sizeof(P));
            }
            for (; done + SPLIT_GRAPH_STEPS <= n_steps; done += SPLIT_GRAPH_STEPS)
                ZDA_CUDA_OK(cudaGraphLaunch(split_exec[which], st));
        }
        for (int n = done; n < n_steps; ++n) {      // the tail (or everything) as plain launches
            P.n = n;
            launch_split_step<T>(P, grd, blk, st);
            launches += per_step;
            int rc = periodic_check<T>(n);
            if (rc != ZDA_OK) return rc;
        }
        launches += (long long)per_step * done;
        return ZDA_OK;
    }
    ~Zone() override {
        for (int w = 0; w < 2; ++w) if (split_exec[w]) cudaGraphExecDestroy(split_exec[w]);
        if (cap_st) cudaStreamDestroy(cap_st);
    }

    int run(int which, int n_steps) {
        return d.complex_fields ? run_T<CR>(which, n_steps) : run_T<R>(which, n_steps);
    }

    int run_forward(int n_steps) override {
        int rc = run(ZDA_FWD, n_steps);
        if (rc == ZDA_OK) { have_fwd = true; have_adj = false; have_src[1] = false; }
        return rc;
    }
    int run_adjoint(int n_steps) override {
        if (!have_src[1]) return fail(ZDA_E_STATE, "zda_run_adjoint needs zda_build_adjoint_source after the forward run");
        int rc = run(ZDA_ADJ, n_steps);
        if (rc == ZDA_OK) have_adj = true;
        return rc;
    }

    // ---- R20: focal weights -------------------------------------------------------------------
    int set_focal_weights(const void* gw, const double* u, int on_host) override {
        if (adj_monitor_dft)
            return fail(ZDA_E_STATE, "the focal weights share their buffer with the adjoint monitor DFT (ZDA_OPT_ADJ_MONITOR_DFT)");
        // dense [f][c][j][Nr] -> planes (f*3 + c) of the monitor-shaped array, pitched rows; pad columns stay 0
        ZDA_CUDA_OK(cudaMemsetAsync(L.dft_mon[1], 0, (size_t)F * 3 * plane * sizeof(CR), st));
        const cudaMemcpyKind kind = on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
        for (int f = 0; f < F; ++f)
            for (int c = 0; c < 2; ++c)
                ZDA_CUDA_OK(cudaMemcpy2DAsync(L.dft_mon[1] + ((size_t)f * 3 + c) * plane, (size_t)pitch * sizeof(CR),
                                              (const CR*)gw + ((size_t)f * 2 + c) * d.Nphi * d.Nr, (size_t)d.Nr * sizeof(CR),
                                              (size_t)d.Nr * sizeof(CR), (size_t)d.Nphi, kind, st));
        for (int f = 0; f < F; ++f) focal_u[f] = u ? u[f] : 1.0;
        have_focal = true;
        have_src[1] = false;
        if (on_host) ZDA_CUDA_OK(cudaStreamSynchronize(st));
        return ZDA_OK;
    }
    // R24: the weights of the on-axis focal point focal_dz above the monitor plane, from the first
    // Rayleigh-Sommerfeld integral; see include/zda.h.  Two small kernels, all in double; the wedge sums (2 Nphi complex
    // doubles) sit in the density map's scratch plane.
    int build_focal_weights(double focal_dz, const double* u) override {
        if (adj_monitor_dft)
            return fail(ZDA_E_STATE, "the focal weights share their buffer with the adjoint monitor DFT (ZDA_OPT_ADJ_MONITOR_DFT)");
        if ((size_t)Nrd * sizeof(R) < 2 * sizeof(Cx<double>))
            return fail(ZDA_E_BADARG, "zda_build_focal_weights needs a design box at least %d cells wide in r", (int)(32 / sizeof(R)));
        Cx<double>* C = reinterpret_cast<Cx<double>*>(L.tmp2d);
        const int n = std::max(d.n_fold, 1);
        wedge_sum_kernel<R><<<(d.Nphi + 63) / 64, 64, 0, st>>>(C, d.Nphi, n, d.dphi, d.Nphi * d.dphi, d.phase_re, d.phase_im);
        FocalK<R> K;
        K.F = F;
        for (int f = 0; f < F; ++f) K.k[f] = omega[f] * std::sqrt(eps_bg[d.monitor_k]);
        ZDA_CUDA_OK(cudaMemsetAsync(L.dft_mon[1], 0, (size_t)F * 3 * plane * sizeof(CR), st));
        focal_weights_kernel<R><<<dim3((d.Nr + 127) / 128, d.Nphi), 128, 0, st>>>(C, L.dft_mon[1], d.Nr, d.Nphi, pitch, d.r_in, d.dr,
                                                                                   d.dr * d.dphi, focal_dz, K);
        launches += 2;
        ZDA_CUDA_OK(cudaGetLastError());
        for (int f = 0; f < F; ++f) focal_u[f] = u ? u[f] : 1.0;
        have_focal = true;
        have_src[1] = false;
        return ZDA_OK;
    }
    bool has_focal_weights() const override { return have_focal; }
    int n_freq() const override { return F; }
    // S_f of the last forward run (synchronises)
    int focal_sums(int m0, int m1, double* S_re, double* S_im) {
        const int nb = N_PARTIAL / (2 * ZDA_MAX_FREQ);
        focal_sum_kernel<R><<<dim3(nb, F), 256, 0, st>>>(L.dft_mon[0], L.dft_mon[1], L.partial, d.Nphi, pitch, m0, m1);
        ++launches;
        ZDA_CUDA_OK(cudaGetLastError());
        std::vector<double> part((size_t)2 * nb * F);
        ZDA_CUDA_OK(cudaMemcpyAsync(part.data(), L.partial, part.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
        ZDA_CUDA_OK(cudaStreamSynchronize(st));
        for (int f = 0; f < F; ++f) {
            S_re[f] = S_im[f] = 0.0;
            for (int b = 0; b < nb; ++b) { S_re[f] += part[((size_t)f * nb + b) * 2]; S_im[f] += part[((size_t)f * nb + b) * 2 + 1]; }
        }
        return ZDA_OK;
    }

    int get_focal_sums(double* S) override {
        if (!have_focal) return fail(ZDA_E_STATE, "zda_get_focal_sums needs zda_set_focal_weights");
        if (!have_fwd) return fail(ZDA_E_STATE, "zda_get_focal_sums needs a forward run");
        double S_re[ZDA_MAX_FREQ], S_im[ZDA_MAX_FREQ];
        int rc = focal_sums(d.npml_r_lo, d.Nr - d.npml_r_hi, S_re, S_im);
        if (rc != ZDA_OK) return rc;
        for (int f = 0; f < F; ++f) { S[2 * f] = S_re[f]; S[2 * f + 1] = S_im[f]; }
        return ZDA_OK;
    }

    // ---- a7: objective + adjoint source ------------------------------------------------------
    int build_adjoint_source(int objective, double t0, double sigma_t, int n_steps, double* F_out,
                             const double* S_total, const double* u_total) override {
        if (!have_fwd) return fail(ZDA_E_STATE, "zda_build_adjoint_source needs a forward run");
        const bool focal = objective == ZDA_OBJ_FOCAL_INTENSITY;
        if (focal && !have_focal) return fail(ZDA_E_STATE, "ZDA_OBJ_FOCAL_INTENSITY needs zda_set_focal_weights");
        if (n_steps > max_steps) return fail(ZDA_E_BADARG, "n_steps %d exceeds max_steps %d", n_steps, max_steps);
        const int m0 = d.npml_r_lo, m1 = d.Nr - d.npml_r_hi;
        // basis pulses q_f(t_{n+1/2}) and their half-step DTFTs qhat_f(w) = dt sum_n q_f e^{i w t}
        std::vector<double> q_re((size_t)F * n_steps), q_im((size_t)F * n_steps);
        for (int f = 0; f < F; ++f)
            for (int n = 0; n < n_steps; ++n) {
                const double t = (n + 0.5) * d.dt, u = t - t0;
                const double env = std::exp(-(u * u) / (2.0 * sigma_t * sigma_t));
                q_re[(size_t)f * n_steps + n] = env * std::cos(omega[f] * u);
                q_im[(size_t)f * n_steps + n] = -env * std::sin(omega[f] * u);
            }
        auto qhat = [&](int f, double w, double& re, double& im) {
            double sr = 0.0, si = 0.0;
            for (int n = 0; n < n_steps; ++n) {
                const double t = (n + 0.5) * d.dt, c = std::cos(w * t), s = std::sin(w * t);
                const double a = q_re[(size_t)f * n_steps + n], b = q_im[(size_t)f * n_steps + n];
                sr += a * c - b * s;
                si += a * s + b * c;
            }
            re = d.dt * sr; im = d.dt * si;
        };
        std::vector<double> V_re(F * F), V_im(F * F), Vm_re(F * F), Vm_im(F * F);
        for (int fp = 0; fp < F; ++fp)
            for (int f = 0; f < F; ++f) {
                qhat(f, omega[fp], V_re[fp * F + f], V_im[fp * F + f]);          // V[f'][f] = qhat_f(w_f')
                double re, im;
                qhat(f, -omega[fp], re, im);
                Vm_re[fp * F + f] = re; Vm_im[fp * F + f] = -im;                  // conj(qhat_f(-w_f'))
            }
        std::vector<R> Minv_h;
        std::vector<double> table;
        int nt;
        if (d.complex_fields) {
            // J = sum_f beta_f q_f(t): a_f' = sum_f V[f'][f] beta_f
            if (!invert_complex(V_re, V_im, F)) return fail(ZDA_E_BADARG, "adjoint pulse matrix is singular");
            Minv_h.resize(2 * F * F);
            for (int t = 0; t < F * F; ++t) { Minv_h[t] = (R)V_re[t]; Minv_h[F * F + t] = (R)V_im[t]; }
            nt = F;
            table.resize((size_t)F * n_steps * 2);
            for (size_t t = 0; t < (size_t)F * n_steps; ++t) { table[2 * t] = q_re[t]; table[2 * t + 1] = q_im[t]; }
        } else {
            // J = Re[sum_f beta_f q_f(t)]: a = P Re(beta) + i M Im(beta), P = (V + Vm)/2, M = (V - Vm)/2
            const int n2 = 2 * F;
            std::vector<double> S((size_t)n2 * n2);
            for (int r = 0; r < F; ++r)
                for (int c = 0; c < F; ++c) {
                    const double Pre = 0.5 * (V_re[r * F + c] + Vm_re[r * F + c]), Pim = 0.5 * (V_im[r * F + c] + Vm_im[r * F + c]);
                    const double Mre = 0.5 * (V_re[r * F + c] - Vm_re[r * F + c]), Mim = 0.5 * (V_im[r * F + c] - Vm_im[r * F + c]);
                    S[(size_t)r * n2 + c] = Pre;        S[(size_t)r * n2 + F + c] = -Mim;
                    S[(size_t)(F + r) * n2 + c] = Pim;  S[(size_t)(F + r) * n2 + F + c] = Mre;
                }
            if (!invert_real(S, n2)) return fail(ZDA_E_BADARG, "adjoint pulse matrix is singular");
            Minv_h.resize((size_t)n2 * n2);
            for (size_t t = 0; t < Minv_h.size(); ++t) Minv_h[t] = (R)S[t];
            nt = n2;
            // Re[beta q] = Re(beta) Re(q) - Im(beta) Im(q): 2F real terms
            table.resize((size_t)n2 * n_steps);
            for (size_t t = 0; t < (size_t)F * n_steps; ++t) { table[t] = q_re[t]; table[(size_t)F * n_steps + t] = -q_im[t]; }
        }
        FocalCoef<R> coef;
        double F_focal = 0.0;
        if (focal) {
            double S_re[ZDA_MAX_FREQ], S_im[ZDA_MAX_FREQ];
            if (S_total) {
                for (int f = 0; f < F; ++f) { S_re[f] = S_total[2 * f]; S_im[f] = S_total[2 * f + 1]; }
            } else {
                int rc = focal_sums(m0, m1, S_re, S_im);
                if (rc != ZDA_OK) return rc;
            }
            for (int f = 0; f < F; ++f) {
                const double uf = S_total ? (u_total ? u_total[f] : 1.0) : focal_u[f];
                coef.c[f] = CR{(R)(uf * S_re[f]), (R)(-uf * S_im[f])};    // u_f conj(S_f)
                F_focal += uf * (S_re[f] * S_re[f] + S_im[f] * S_im[f]);
            }
        }
        const CR* gw = focal ? L.dft_mon[1] : nullptr;
        ZDA_CUDA_OK(cudaMemcpyAsync(L.Minv, Minv_h.data(), Minv_h.size() * sizeof(R), cudaMemcpyHostToDevice, st));
        const dim3 grid((pitch + 127) / 128, d.Nphi);
        if (d.complex_fields)
            adjoint_source_kernel<CR><<<grid, 128, 0, st>>>(L.dft_mon[0], (CR*)L.A[1][0], (CR*)L.A[1][1], L.Minv, d.Nr,
                                                            d.Nphi, pitch, F, m0, m1, gw, L.rc, coef);
        else
            adjoint_source_kernel<R><<<grid, 128, 0, st>>>(L.dft_mon[0], (R*)L.A[1][0], (R*)L.A[1][1], L.Minv, d.Nr,
                                                           d.Nphi, pitch, F, m0, m1, gw, L.rc, coef);
        ++launches;
        ZDA_CUDA_OK(cudaGetLastError());
        int rc = upload_table(1, nt, table.data(), n_steps);   // synchronises (Minv_h stays alive until here)
        if (rc != ZDA_OK) return rc;
        if (F_out && focal) {
            *F_out = F_focal;
        } else if (F_out) {
            objective_kernel<R><<<N_PARTIAL, 256, 0, st>>>(L.dft_mon[0], L.rc, L.partial, d.Nr, d.Nphi, pitch, F, m0, m1);
            ++launches;
            ZDA_CUDA_OK(cudaGetLastError());
            std::vector<double> part(N_PARTIAL);
            ZDA_CUDA_OK(cudaMemcpyAsync(part.data(), L.partial, N_PARTIAL * sizeof(double), cudaMemcpyDeviceToHost, st));
            ZDA_CUDA_OK(cudaStreamSynchronize(st));
            double s = 0.0;
            for (double v : part) s += v;
            *F_out = s;
        }
        return ZDA_OK;
    }

    // ---- outputs ---------------------------------------------------------------------------
    int get_dft(int which, int region, int comp, int freq, void* out, int on_host) override {
        if (which != ZDA_FWD && which != ZDA_ADJ) return fail(ZDA_E_BADARG, "which must be ZDA_FWD or ZDA_ADJ");
        if (comp < 0 || comp > 2 || freq < 0 || freq >= F) return fail(ZDA_E_BADARG, "comp/freq out of range");
        if ((which == ZDA_FWD && !have_fwd) || (which == ZDA_ADJ && !have_adj)) return fail(ZDA_E_STATE, "that run has not been made");
        const cudaMemcpyKind kind = on_host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
        if (region == ZDA_DESIGN) {
            const CR* src = L.dft_design[which] + ((size_t)freq * 3 + comp) * Ld * plane + d.design_i0;
            ZDA_CUDA_OK(cudaMemcpy2DAsync(out, (size_t)Nrd * sizeof(CR), src, (size_t)pitch * sizeof(CR), (size_t)Nrd * sizeof(CR),
                                          (size_t)Ld * d.Nphi, kind, st));
        } else if (region == ZDA_MONITOR) {
            if (which == ZDA_ADJ && !adj_monitor_dft) return fail(ZDA_E_STATE, "adjoint monitor DFT is off (ZDA_OPT_ADJ_MONITOR_DFT)");
            const CR* src = L.dft_mon[which] + ((size_t)freq * 3 + comp) * plane;
            ZDA_CUDA_OK(cudaMemcpy2DAsync(out, (size_t)d.Nr * sizeof(CR), src, (size_t)pitch * sizeof(CR), (size_t)d.Nr * sizeof(CR),
                                          (size_t)d.Nphi, kind, st));
        } else {
            return fail(ZDA_E_BADARG, "region must be ZDA_DESIGN or ZDA_MONITOR");
        }
        if (on_host) ZDA_CUDA_OK(cudaStreamSynchronize(st));
        return ZDA_OK;
    }

    int get_field(int comp, void* out, int on_host) override {
        if (comp < 0 || comp > 5) return fail(ZDA_E_BADARG, "comp out of range");
        char* src = comp < 3 ? L.E[cur][comp] : L.H[cur][comp - 3];
        // [Nz][Nphi + 2 FIELD_GHOST][pitch] with ghost rows -> dense [Nz][Nphi][Nr]
        cudaMemcpy3DParms cp;
        std::memset(&cp, 0, sizeof(cp));
        cp.srcPtr = make_cudaPitchedPtr(src, (size_t)pitch * es, (size_t)pitch * es, (size_t)d.Nphi + 2 * field_ghost(d));
        cp.srcPos = make_cudaPos(0, field_ghost(d), 0);
        cp.dstPtr = make_cudaPitchedPtr(out, (size_t)d.Nr * es, (size_t)d.Nr * es, (size_t)d.Nphi);
        cp.extent = make_cudaExtent((size_t)d.Nr * es, (size_t)d.Nphi, (size_t)d.Nz);
        cp.kind = on_host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
        ZDA_CUDA_OK(cudaMemcpy3DAsync(&cp, st));
        if (on_host) ZDA_CUDA_OK(cudaStreamSynchronize(st));
        return ZDA_OK;
    }

    int gradient(void* dF_deps, void* dF_deps_zsum, void* dF_drho, int on_host) override {
        if (!have_fwd || !have_adj) return fail(ZDA_E_STATE, "zda_gradient needs a forward and an adjoint run");
        if (dF_drho && !have_density) return fail(ZDA_E_STATE, "dF_drho needs zda_set_density");
        const size_t n2 = (size_t)Nrd * d.Nphi, n3 = n2 * Ld;
        GradParams<R> G;
        G.F = F;
        for (int f = 0; f < F; ++f) G.Omega[f] = (R)((2.0 / d.dt) * std::sin(omega[f] * d.dt / 2.0));
        R* box = nullptr;
        if (dF_deps) box = on_host ? L.staging : (R*)dF_deps;
        R* zs = L.g2d;
        if (dF_deps_zsum && !on_host) zs = (R*)dF_deps_zsum;
        const dim3 grid((Nrd + 127) / 128, d.Nphi);
        gradient_kernel<R><<<grid, 128, 0, st>>>(L.dft_design[0], L.dft_design[1], L.rc, box, zs, Nrd, d.Nphi, Ld, pitch,
                                                 d.design_i0, G);
        ++launches;
        ZDA_CUDA_OK(cudaGetLastError());
        if (dF_deps && on_host) ZDA_CUDA_OK(cudaMemcpyAsync(dF_deps, L.staging, n3 * sizeof(R), cudaMemcpyDeviceToHost, st));
        if (dF_deps_zsum && on_host) ZDA_CUDA_OK(cudaMemcpyAsync(dF_deps_zsum, zs, n2 * sizeof(R), cudaMemcpyDeviceToHost, st));
        if (dF_drho) {
            // a2 VJP: x (eps_h - eps0) x projection derivative, then the transposed filter (phi first, then r)
            project_vjp_kernel<R><<<(int)((n2 + 255) / 256), 256, 0, st>>>(zs, L.rho_f, L.tmp2d, (int)n2, (R)dens_eps0,
                                                                          (R)dens_eps_h, (R)dens_beta, (R)dens_eta);
            R* dst = on_host ? L.tmp2d : (R*)dF_drho;
            if (dens_conic_radius > 0.0) {
                // transpose of the normalised cone: divide by the output cell's weight sum, then the symmetric stencil
                const ConicP<R> C = conic_params(dens_conic_radius);
                conic_kernel<R, 1><<<grid, 128, 0, st>>>(L.tmp2d, L.rho, Nrd, d.Nphi, C);
                conic_kernel<R, 2><<<grid, 128, 0, st>>>(L.rho, dst, Nrd, d.Nphi, C);
            } else {
                const FilterW<R> W = filter_weights(dens_sigma);
                // the periodic phi filter with symmetric weights is its own transpose
                filter_phi_kernel<R><<<grid, 128, 0, st>>>(L.tmp2d, L.rho, Nrd, d.Nphi, W);
                filter_r_T_kernel<R><<<grid, 128, 0, st>>>(L.rho, dst, Nrd, d.Nphi, W);
            }
            launches += 3;
            ZDA_CUDA_OK(cudaGetLastError());
            if (on_host) ZDA_CUDA_OK(cudaMemcpyAsync(dF_drho, dst, n2 * sizeof(R), cudaMemcpyDeviceToHost, st));
        }
        if (on_host) ZDA_CUDA_OK(cudaStreamSynchronize(st));
        return ZDA_OK;
    }

    int check_finite() override {
        double total = 0.0;
        for (int c = 0; c < 3; ++c) {
            if (d.complex_fields) nonfinite_kernel<CR><<<N_PARTIAL, 256, 0, st>>>((const CR*)L.E[cur][c], fvol, L.partial);
            else nonfinite_kernel<R><<<N_PARTIAL, 256, 0, st>>>((const R*)L.E[cur][c], fvol, L.partial);
            ++launches;
            ZDA_CUDA_OK(cudaGetLastError());
            std::vector<double> part(N_PARTIAL);
            ZDA_CUDA_OK(cudaMemcpyAsync(part.data(), L.partial, N_PARTIAL * sizeof(double), cudaMemcpyDeviceToHost, st));
            ZDA_CUDA_OK(cudaStreamSynchronize(st));
            for (double v : part) total += v;
        }
        if (total > 0.0) return fail(ZDA_E_NAN, "%.0f non-finite E values", total);
        return ZDA_OK;
    }
};

template <class R> size_t workspace_bytes_impl(const zda_zone_desc& d, int max_steps) {
    Arena ar;
    ZoneLayout<R> L;
    carve<R>(d, max_steps, (d.Nr + 31) / 32 * 32, ar, L);
    return ar.off;
}

template <class R>
int create_zone_impl(const zda_zone_desc& d, const double* eps_bg_z, int max_steps, void* ws, size_t bytes,
                     cudaStream_t stream, ZoneBase** out) {
    Zone<R>* z = new Zone<R>(d, stream, max_steps);
    int rc = z->init(eps_bg_z, ws, bytes);
    if (rc != ZDA_OK) { delete z; return rc; }
    *out = z;
    return ZDA_OK;
}

}  // namespace zda
