// Split time-loop kernels: one H-update pass and one E-update pass per step (a3, a4 of
// SURVEY 8a), one thread per voxel, r along threadIdx.x (coalesced).  CPML, phi wrap,
// source sheet and running DFT are fused into the two passes.  This is the reference
// GPU path: it covers every feature (axis zones included) in both precisions.
#pragma once
#include <cooperative_groups.h>
#include "zda_device.cuh"
#include "zda_common.h"

namespace zda {

constexpr int SPLIT_BX = 64, SPLIT_BY = 4, SPLIT_BZ = 2;

// H update of voxel (i, j, k), in place (a3)
template <class T>
__device__ __forceinline__ void h_update_at(const StepParams<T>& P, const int i, const int j, const int k) {
    using R = typename ElemTraits<T>::Real;
    const size_t row = (size_t)P.pitch;
    const size_t plane = row * P.Nphi, fplane = P.fplane;
    const size_t c = (size_t)k * fplane + (size_t)(j + P.ghost) * row + i;
    const bool wrap = (j + 1 == P.Nphi);
    const size_t cjp = wrap ? c - (size_t)j * row : c + row;

    HIn<T, R> in;
    in.er = P.E[0][c]; in.ep = P.E[1][c]; in.ez = P.E[2][c];
    in.er_jp = P.E[0][cjp]; in.ez_jp = P.E[2][cjp];
    if (wrap) { in.er_jp = phase_mul(P.pr, P.pi, in.er_jp); in.ez_jp = phase_mul(P.pr, P.pi, in.ez_jp); }
    const bool kin = (k + 1 < P.Nz), iin = (i + 1 < P.Nr);
    in.er_kp = kin ? P.E[0][c + fplane] : zero_of<T>();
    in.ep_kp = kin ? P.E[1][c + fplane] : zero_of<T>();
    in.ep_ip = iin ? P.E[1][c + 1] : zero_of<T>();
    in.ez_ip = iin ? P.E[2][c + 1] : zero_of<T>();
    const R* rc = P.rc;
    in.inv_rdphi_int = rc[RC_INV_RDPHI_INT * P.pitch + i];
    in.inv_rdphi_half = rc[RC_INV_RDPHI_HALF * P.pitch + i];
    in.ca = rc[RC_CA * P.pitch + i];
    in.cb = rc[RC_CB * P.pitch + i];
    in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.dt = P.dt;
    in.skip_hr = (P.has_axis && i == 0);

    // CPML slabs (auxiliaries exist only there)
    const int npz = P.npz_lo + P.npz_hi, npr = P.npr_lo + P.npr_hi;
    int kz = -1, ir = -1;
    if (k < P.npz_lo) kz = k; else if (k >= P.Nz - P.npz_hi) kz = P.npz_lo + (k - (P.Nz - P.npz_hi));
    if (i < P.npr_lo) ir = i; else if (i >= P.Nr - P.npr_hi) ir = P.npr_lo + (i - (P.Nr - P.npr_hi));
    in.zs = kz >= 0; in.rs = ir >= 0;
    (void)npz;
    size_t cz_ = 0, cr_ = 0;
    T p0 = zero_of<T>(), p1 = zero_of<T>(), p2 = zero_of<T>(), p3 = zero_of<T>();
    in.bz = in.cz = in.br = in.cr = R(0); in.ikz = in.ikr = R(1);
    if (in.zs) {
        cz_ = (size_t)kz * plane + (size_t)j * row + i;
        p0 = P.psiH_z[0][cz_]; p1 = P.psiH_z[1][cz_];
        in.bz = P.zc[ZC_B_H * P.Nz + k]; in.cz = P.zc[ZC_C_H * P.Nz + k]; in.ikz = P.zc[ZC_IK_H * P.Nz + k];
    }
    if (in.rs) {
        cr_ = ((size_t)k * P.Nphi + j) * npr + ir;
        p2 = P.psiH_r[0][cr_]; p3 = P.psiH_r[1][cr_];
        in.br = rc[RC_B_H * P.pitch + i]; in.cr = rc[RC_C_H * P.pitch + i]; in.ikr = rc[RC_IK_H * P.pitch + i];
    }
    // R25: exact complex-r form in the outer r-slab
    T q0 = zero_of<T>(), q1 = zero_of<T>();
    in.xr = P.rpml_exact && (i >= P.Nr - P.npr_hi);
    if (in.xr) {
        q0 = P.chiH[0][cr_]; q1 = P.chiH[1][cr_];
        in.bq_i = rc[RC_BQ_I * P.pitch + i]; in.cq_i = rc[RC_CQ_I * P.pitch + i];
        in.bq_h = rc[RC_BQ_H * P.pitch + i]; in.cq_h = rc[RC_CQ_H * P.pitch + i]; in.hir = rc[RC_HIR_H * P.pitch + i];
    }
    T hr = P.H[0][c], hp = P.H[1][c], hz = P.H[2][c];
    h_update_voxel(in, hr, hp, hz, p0, p1, p2, p3, q0, q1);
    P.H[0][c] = hr; P.H[1][c] = hp; P.H[2][c] = hz;
    if (in.zs) { P.psiH_z[0][cz_] = p0; P.psiH_z[1][cz_] = p1; }
    if (in.rs) { P.psiH_r[0][cr_] = p2; P.psiH_r[1][cr_] = p3; }
    if (in.xr) { P.chiH[0][cr_] = q0; P.chiH[1][cr_] = q1; }
}

template <class T>
__global__ void __launch_bounds__(SPLIT_BX * SPLIT_BY * SPLIT_BZ)
h_update_kernel(const __grid_constant__ StepParams<T> P) {
    const int i = blockIdx.x * SPLIT_BX + threadIdx.x;
    const int j = blockIdx.y * SPLIT_BY + threadIdx.y;
    const int k = blockIdx.z * SPLIT_BZ + threadIdx.z;
    // device-side step counter (graph replay): this kernel opens step n; nothing reads the counter while it runs
    if (P.n_dev && i == 0 && j == 0 && k == 0) *const_cast<int*>(P.n_dev) += 1;
    if (i >= P.Nr || j >= P.Nphi || k >= P.Nz) return;
    h_update_at<T>(P, i, j, k);
}

// mean_j Hphi[0, j, k] for the axis loop integral (R4); one thread per k, ascending j.
template <class T>
__global__ void axis_mean_kernel(const __grid_constant__ StepParams<T> P, T* out) {
    using R = typename ElemTraits<T>::Real;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= P.Nz) return;
    const size_t row = (size_t)P.pitch;
    T sum = zero_of<T>();
    for (int j = 0; j < P.Nphi; ++j) sum = sum + P.H[1][(size_t)k * P.fplane + (size_t)(j + P.ghost) * row];
    // mean = sum / Nphi (a true division, as the definition is written)
    if constexpr (ElemTraits<T>::cplx) out[k] = T{sum.x / R(P.Nphi), sum.y / R(P.Nphi)};
    else out[k] = sum / R(P.Nphi);
}

// E update of voxel (i, j, k) of step n_step, in place (a4-a6); axis_mean_k = mean_j Hphi[0, j, k] (axis zones, i == 0)
template <class T>
__device__ __forceinline__ void e_update_at(const StepParams<T>& P, const int i, const int j, const int k, const int n_step,
                                            const T axis_mean_k) {
    using R = typename ElemTraits<T>::Real;
    const size_t row = (size_t)P.pitch;
    const size_t plane = row * P.Nphi, fplane = P.fplane;
    const size_t pj = (size_t)j * row + i;
    const size_t c = (size_t)k * fplane + P.ghost * row + pj;
    const bool wrap = (j == 0);
    const size_t cjm = wrap ? c + (size_t)(P.Nphi - 1) * row : c - row;

    EIn<T, R> in;
    in.hr = P.H[0][c]; in.hp = P.H[1][c]; in.hz = P.H[2][c];
    in.hr_jm = P.H[0][cjm]; in.hz_jm = P.H[2][cjm];
    if (wrap) { in.hr_jm = phase_mul(P.pr, -P.pi, in.hr_jm); in.hz_jm = phase_mul(P.pr, -P.pi, in.hz_jm); }
    in.k_pos = (k > 0); in.i_pos = (i > 0);
    in.hr_km = in.k_pos ? P.H[0][c - fplane] : zero_of<T>();
    in.hp_km = in.k_pos ? P.H[1][c - fplane] : zero_of<T>();
    in.hp_im = in.i_pos ? P.H[1][c - 1] : zero_of<T>();
    in.hz_im = in.i_pos ? P.H[2][c - 1] : zero_of<T>();
    const R* rc = P.rc;
    in.inv_rdphi_int = rc[RC_INV_RDPHI_INT * P.pitch + i];
    in.inv_rdphi_half = rc[RC_INV_RDPHI_HALF * P.pitch + i];
    in.cc = rc[RC_CC * P.pitch + i];
    in.cd = rc[RC_CD * P.pitch + i];
    in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz;
    const bool in_mat = (k >= P.mk0 && k < P.mk1);
    in.cE = in_mat ? P.cE_design[(size_t)(k - P.mk0) * plane + pj] : P.zc[ZC_CE_BG * P.Nz + k];

    // current sheet J = sum_q A_q s_q[n] on plane src_k
    in.jr = zero_of<T>(); in.jp = zero_of<T>();
    if (k == P.src_k && P.n_terms > 0 && n_step < P.tab_len) {
        for (int q = 0; q < P.n_terms; ++q) {
            const T s = P.s_tab[(size_t)q * P.tab_len + n_step];
            const T ar = P.A_r[(size_t)q * plane + pj], ap = P.A_phi[(size_t)q * plane + pj];
            if constexpr (ElemTraits<T>::cplx) { in.jr = in.jr + cmul(s, ar); in.jp = in.jp + cmul(s, ap); }
            else { in.jr = in.jr + s * ar; in.jp = in.jp + s * ap; }
        }
    }

    const int npr = P.npr_lo + P.npr_hi;
    int kz = -1, ir = -1;
    if (k < P.npz_lo) kz = k; else if (k >= P.Nz - P.npz_hi) kz = P.npz_lo + (k - (P.Nz - P.npz_hi));
    if (i < P.npr_lo) ir = i; else if (i >= P.Nr - P.npr_hi) ir = P.npr_lo + (i - (P.Nr - P.npr_hi));
    in.zs = kz >= 0; in.rs = ir >= 0;
    size_t cz_ = 0, cr_ = 0;
    T p0 = zero_of<T>(), p1 = zero_of<T>(), p2 = zero_of<T>(), p3 = zero_of<T>();
    in.bz = in.cz = in.br = in.cr = R(0); in.ikz = in.ikr = R(1);
    if (in.zs) {
        cz_ = (size_t)kz * plane + pj;
        p0 = P.psiE_z[0][cz_]; p1 = P.psiE_z[1][cz_];
        in.bz = P.zc[ZC_B_I * P.Nz + k]; in.cz = P.zc[ZC_C_I * P.Nz + k]; in.ikz = P.zc[ZC_IK_I * P.Nz + k];
    }
    if (in.rs) {
        cr_ = ((size_t)k * P.Nphi + j) * npr + ir;
        p2 = P.psiE_r[0][cr_]; p3 = P.psiE_r[1][cr_];
        in.br = rc[RC_B_I * P.pitch + i]; in.cr = rc[RC_C_I * P.pitch + i]; in.ikr = rc[RC_IK_I * P.pitch + i];
    }
    T q0 = zero_of<T>(), q1 = zero_of<T>();
    in.xr = P.rpml_exact && (i >= P.Nr - P.npr_hi);
    if (in.xr) {
        q0 = P.chiE[0][cr_]; q1 = P.chiE[1][cr_];
        in.bq_i = rc[RC_BQ_I * P.pitch + i]; in.cq_i = rc[RC_CQ_I * P.pitch + i];
        in.bq_h = rc[RC_BQ_H * P.pitch + i]; in.cq_h = rc[RC_CQ_H * P.pitch + i]; in.hir = rc[RC_HIR_I * P.pitch + i];
    }
    T er = P.E[0][c], ep = P.E[1][c], ez = P.E[2][c];
    e_update_voxel(in, er, ep, ez, p0, p1, p2, p3, q0, q1);
    // R4: on-axis Ez from Ampere's law on the circle r = dr/2 (one unknown per k, replicated over j)
    if (P.has_axis && i == 0 && P.p_is_one) {
        const R cEa = P.zc[ZC_CE_AXIS * P.Nz + k];
        ez = ez + cEa * ((R(4) * P.inv_dr) * axis_mean_k);
    }
    P.E[0][c] = er; P.E[1][c] = ep; P.E[2][c] = ez;
    if (in.zs) { P.psiE_z[0][cz_] = p0; P.psiE_z[1][cz_] = p1; }
    if (in.rs) { P.psiE_r[0][cr_] = p2; P.psiE_r[1][cr_] = p3; }
    if (in.xr) { P.chiE[0][cr_] = q0; P.chiE[1][cr_] = q1; }

    // running DFT (R8): Ehat_{c,f} += tw_f E_c^{n+1}
    const bool in_design = (k >= P.dk0 && k < P.dk1 && i >= P.di0 && i < P.di1);
    if (in_design || k == P.mon_k) {
        const int Ld = P.dk1 - P.dk0;
        for (int f = 0; f < P.F; ++f) {
            const Cx<R> tw = P.tw[(size_t)n_step * P.F + f];
            const Cx<R> a0 = tw_mul(tw, er), a1 = tw_mul(tw, ep), a2 = tw_mul(tw, ez);
            if (in_design) {
                Cx<R>* d = P.dft_design + ((size_t)f * 3 * Ld + (k - P.dk0)) * plane + pj;
                d[0] = d[0] + a0;
                d[(size_t)Ld * plane] = d[(size_t)Ld * plane] + a1;
                d[(size_t)2 * Ld * plane] = d[(size_t)2 * Ld * plane] + a2;
            }
            if (k == P.mon_k && P.dft_mon) {
                Cx<R>* m = P.dft_mon + (size_t)f * 3 * plane + pj;
                m[0] = m[0] + a0;
                m[plane] = m[plane] + a1;
                m[2 * plane] = m[2 * plane] + a2;
            }
        }
    }
}

template <class T>
__global__ void __launch_bounds__(SPLIT_BX * SPLIT_BY * SPLIT_BZ)
e_update_kernel(const __grid_constant__ StepParams<T> P) {
    const int n_step = P.n_dev ? *P.n_dev : P.n;
    const int i = blockIdx.x * SPLIT_BX + threadIdx.x;
    const int j = blockIdx.y * SPLIT_BY + threadIdx.y;
    const int k = blockIdx.z * SPLIT_BZ + threadIdx.z;
    if (i >= P.Nr || j >= P.Nphi || k >= P.Nz) return;
    e_update_at<T>(P, i, j, k, n_step, (P.has_axis && i == 0 && P.p_is_one) ? P.axis_mean[k] : zero_of<T>());
}

// Small zones (the paper's continuously axisymmetric first zone: 2e5 voxels): ONE persistent cooperative
// kernel makes all the time steps of a run; the H and E passes are separated by grid-wide barriers instead of kernel
// boundaries, and the whole state (fields + auxiliaries, a few MB) stays in L2.  Same per-voxel functions as the split
// kernels, so the results are bit-identical to theirs.  The axis loop integral's phi-mean (R4) is taken by the thread
// that needs it (ascending j, as axis_mean_kernel does).
constexpr int PERSIST_THREADS = 512;       // one block per SM: the grid barrier then spans 148 blocks
template <class T>
__global__ void __launch_bounds__(PERSIST_THREADS)
persist_kernel(const __grid_constant__ StepParams<T> P, const int n0, const int n_steps) {
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();     // launched with cudaLaunchCooperativeKernel
    using R = typename ElemTraits<T>::Real;
    const long n_vox = (long)P.Nr * P.Nphi * P.Nz;
    const long tid0 = (long)blockIdx.x * blockDim.x + threadIdx.x, stride = (long)gridDim.x * blockDim.x;
    for (int n = n0; n < n0 + n_steps; ++n) {
        for (long t = tid0; t < n_vox; t += stride) {
            const int i = (int)(t % P.Nr), j = (int)((t / P.Nr) % P.Nphi), k = (int)(t / ((long)P.Nr * P.Nphi));
            h_update_at<T>(P, i, j, k);
        }
        grid.sync();
        for (long t = tid0; t < n_vox; t += stride) {
            const int i = (int)(t % P.Nr), j = (int)((t / P.Nr) % P.Nphi), k = (int)(t / ((long)P.Nr * P.Nphi));
            T mean = zero_of<T>();
            if (P.has_axis && i == 0 && P.p_is_one) {
                T sum = zero_of<T>();
                for (int jj = 0; jj < P.Nphi; ++jj) sum = sum + P.H[1][(size_t)k * P.fplane + (size_t)(jj + P.ghost) * P.pitch];
                if constexpr (ElemTraits<T>::cplx) mean = T{sum.x / R(P.Nphi), sum.y / R(P.Nphi)};
                else mean = sum / R(P.Nphi);
            }
            e_update_at<T>(P, i, j, k, n, mean);
        }
        grid.sync();
    }
}

}  // namespace zda
