// Device-side building blocks shared by the split and the fused time-loop kernels:
// element types, the CPML operator, and the per-voxel H and E updates (Eq. 3-5,
// PAPER.md:53-62; discrete form DESIGN.md "Update equations").
//
// Every expression is written in the order DESIGN.md fixes (difference, times its 1-D
// coefficient, CPML, bracket left to right, then the update), so that the fp64 build
// (compiled with -fmad=false) evaluates exactly what is written.
#pragma once
#include <cuda_runtime.h>

namespace zda {

// complex element: interleaved (re, im), aligned for one vector load
template <class Real> struct alignas(2 * sizeof(Real)) Cx {
    Real x, y;
};

template <class Real> __host__ __device__ __forceinline__ Cx<Real> operator+(Cx<Real> a, Cx<Real> b) { return {a.x + b.x, a.y + b.y}; }
template <class Real> __host__ __device__ __forceinline__ Cx<Real> operator-(Cx<Real> a, Cx<Real> b) { return {a.x - b.x, a.y - b.y}; }
template <class Real> __host__ __device__ __forceinline__ Cx<Real> operator*(Cx<Real> a, Real s) { return {a.x * s, a.y * s}; }
template <class Real> __host__ __device__ __forceinline__ Cx<Real> operator*(Real s, Cx<Real> a) { return {s * a.x, s * a.y}; }
template <class Real> __host__ __device__ __forceinline__ Cx<Real> cmul(Cx<Real> a, Cx<Real> b) {
    return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x};
}

template <class T> struct ElemTraits;
template <> struct ElemTraits<float> { using Real = float; static constexpr bool cplx = false; };
template <> struct ElemTraits<double> { using Real = double; static constexpr bool cplx = false; };
template <class R> struct ElemTraits<Cx<R>> { using Real = R; static constexpr bool cplx = true; };

template <class T> __host__ __device__ __forceinline__ T zero_of() { return T{}; }

// phase multiply p * X (phi-boundary wrap, Eq. 1-2)
__device__ __forceinline__ float phase_mul(float pr, float, float x) { return pr * x; }
__device__ __forceinline__ double phase_mul(double pr, double, double x) { return pr * x; }
template <class R> __device__ __forceinline__ Cx<R> phase_mul(R pr, R pi, Cx<R> x) {
    return {pr * x.x - pi * x.y, pr * x.y + pi * x.x};
}

// twiddle multiply tw * E for the running DFT (R8): complex x real or complex x complex
template <class R> __device__ __forceinline__ Cx<R> tw_mul(Cx<R> tw, R e) { return {tw.x * e, tw.y * e}; }
template <class R> __device__ __forceinline__ Cx<R> tw_mul(Cx<R> tw, Cx<R> e) { return cmul(tw, e); }

// CPML operator (R5): psi <- b psi + c D evaluated before use; P[D] = D / kappa + psi
template <class T, class R> __device__ __forceinline__ T cpml_apply(T D, T& psi, R b, R c, R ik) {
    psi = b * psi + c * D;
    return D * ik + psi;
}

// Per-voxel H update (Faraday, Eq. 3 with the curl of Eq. 5).  E neighbours carry their ghosts
// (PEC zeros in r, z; phase-wrapped in phi) already.  psi* are updated in place (registers);
// zs / rs say whether this voxel lies in a z- / r-slab (else psi is identically 0, kappa = 1).
template <class T, class R> struct HIn {
    T er, ep, ez;          // E at (i, j, k)
    T er_jp, ez_jp;        // at j + 1
    T er_kp, ep_kp;        // at k + 1
    T ep_ip, ez_ip;        // at i + 1
    R inv_rdphi_int, inv_rdphi_half, ca, cb;
    R inv_dr, inv_dz, dt;
    R bz, cz, ikz, br, cr, ikr;   // CPML at (k + 1/2), (i + 1/2)
    bool zs, rs, skip_hr;
    // R25, exact cylindrical PML in the outer r-slab: xr marks its cells; (bq, cq) are the coefficients of the 1/r~
    // operator at i (Hr) and at i + 1/2 (Hz), hir = 1 / (2 r_{i+1/2})
    bool xr = false;
    R bq_i = R(0), cq_i = R(0), bq_h = R(0), cq_h = R(0), hir = R(0);
};

// The skipped (PEC / axis) components are computed and then discarded by a select, so that the compiler emits
// straight-line code instead of a divergence region per component.
template <class T, class R>
__device__ __forceinline__ void h_update_voxel(const HIn<T, R>& in, T& hr, T& hp, T& hz,
                                               T& psi_hr_z, T& psi_hp_z, T& psi_hp_r, T& psi_hz_r, T& chi_hr, T& chi_hz) {
    {
        T psi = psi_hr_z, chi = chi_hr;
        T t1 = (in.ez_jp - in.ez) * in.inv_rdphi_int;
        if (in.xr) t1 = cpml_apply(t1, chi, in.bq_i, in.cq_i, R(1));          // (1 / r~) d_phi Ez
        const T Dz = (in.ep_kp - in.ep) * in.inv_dz;
        const T t2 = in.zs ? cpml_apply(Dz, psi, in.bz, in.cz, in.ikz) : Dz;
        const T v = hr - in.dt * (t1 - t2);
        if (!in.skip_hr) { hr = v; psi_hr_z = psi; chi_hr = chi; }
    }
    {
        const T Dz = (in.er_kp - in.er) * in.inv_dz;
        const T t1 = in.zs ? cpml_apply(Dz, psi_hp_z, in.bz, in.cz, in.ikz) : Dz;
        const T Dr = (in.ez_ip - in.ez) * in.inv_dr;
        const T t2 = in.rs ? cpml_apply(Dr, psi_hp_r, in.br, in.cr, in.ikr) : Dr;
        hp = hp - in.dt * (t1 - t2);
    }
    if (!in.xr) {
        const T Dr = in.ep_ip * in.ca - in.ep * in.cb;
        const T t1 = in.rs ? cpml_apply(Dr, psi_hz_r, in.br, in.cr, in.ikr) : Dr;
        const T t2 = (in.er_jp - in.er) * in.inv_rdphi_half;
        hz = hz - in.dt * (t1 - t2);
    } else {
        // (1/(r~ s_r)) d_r(r~ Ephi) - (1/r~) d_phi Er = (1/s_r) d_r Ephi + (1/r~)[Ephi - d_phi Er]   (d r~/dr = s_r)
        const T Dr = (in.ep_ip - in.ep) * in.inv_dr;
        const T t1 = cpml_apply(Dr, psi_hz_r, in.br, in.cr, in.ikr);
        const T q = (in.ep_ip + in.ep) * in.hir - (in.er_jp - in.er) * in.inv_rdphi_half;
        const T t2 = cpml_apply(q, chi_hz, in.bq_h, in.cq_h, R(1));
        hz = hz - in.dt * (t1 + t2);
    }
}
// the quasi-CPML only (callers without the R25 auxiliaries)
template <class T, class R>
__device__ __forceinline__ void h_update_voxel(const HIn<T, R>& in, T& hr, T& hp, T& hz,
                                               T& psi_hr_z, T& psi_hp_z, T& psi_hp_r, T& psi_hz_r) {
    T c0 = zero_of<T>(), c1 = zero_of<T>();
    h_update_voxel(in, hr, hp, hz, psi_hr_z, psi_hp_z, psi_hp_r, psi_hz_r, c0, c1);
}

// Per-voxel E update (Ampere, Eq. 4 with Eq. 5), PEC predicates included (R7):
// Er skipped at k = 0; Ephi skipped at k = 0 or i = 0; Ez skipped at i = 0 (annulus wall;
// the axis value is set by the caller from the loop integral, R4).
template <class T, class R> struct EIn {
    T hr, hp, hz;          // H at (i, j, k)
    T hr_jm, hz_jm;        // at j - 1
    T hr_km, hp_km;        // at k - 1
    T hp_im, hz_im;        // at i - 1
    T jr, jp;              // current sheet (0 off the source plane)
    R inv_rdphi_int, inv_rdphi_half, cc, cd;
    R inv_dr, inv_dz, cE;
    R bz, cz, ikz, br, cr, ikr;   // CPML at k, i
    bool zs, rs, k_pos, i_pos;
    // R25: coefficients of the 1/r~ operator at i + 1/2 (Er) and at i (Ez), hir = 1 / (2 r_i)
    bool xr = false;
    R bq_i = R(0), cq_i = R(0), bq_h = R(0), cq_h = R(0), hir = R(0);
};

template <class T, class R>
__device__ __forceinline__ void e_update_voxel(const EIn<T, R>& in, T& er, T& ep, T& ez,
                                               T& psi_er_z, T& psi_ep_z, T& psi_ep_r, T& psi_ez_r, T& chi_er, T& chi_ez) {
    {
        T psi = psi_er_z, chi = chi_er;
        T t1 = (in.hz - in.hz_jm) * in.inv_rdphi_half;
        if (in.xr) t1 = cpml_apply(t1, chi, in.bq_h, in.cq_h, R(1));          // (1 / r~) d_phi Hz
        const T Dz = (in.hp - in.hp_km) * in.inv_dz;
        const T t2 = in.zs ? cpml_apply(Dz, psi, in.bz, in.cz, in.ikz) : Dz;
        const T v = er + in.cE * (t1 - t2 - in.jr);
        if (in.k_pos) { er = v; psi_er_z = psi; chi_er = chi; }
    }
    {
        T psiz = psi_ep_z, psir = psi_ep_r;
        const T Dz = (in.hr - in.hr_km) * in.inv_dz;
        const T t1 = in.zs ? cpml_apply(Dz, psiz, in.bz, in.cz, in.ikz) : Dz;
        const T Dr = (in.hz - in.hz_im) * in.inv_dr;
        const T t2 = in.rs ? cpml_apply(Dr, psir, in.br, in.cr, in.ikr) : Dr;
        const T v = ep + in.cE * (t1 - t2 - in.jp);
        if (in.k_pos && in.i_pos) { ep = v; psi_ep_z = psiz; psi_ep_r = psir; }
    }
    if (!in.xr) {
        T psi = psi_ez_r;
        const T Dr = in.hp * in.cc - in.hp_im * in.cd;
        const T t1 = in.rs ? cpml_apply(Dr, psi, in.br, in.cr, in.ikr) : Dr;
        const T t2 = (in.hr - in.hr_jm) * in.inv_rdphi_int;
        const T v = ez + in.cE * (t1 - t2);
        if (in.i_pos) { ez = v; psi_ez_r = psi; }
    } else {                                  // the outer slab never holds i = 0
        const T Dr = (in.hp - in.hp_im) * in.inv_dr;
        const T t1 = cpml_apply(Dr, psi_ez_r, in.br, in.cr, in.ikr);
        const T q = (in.hp + in.hp_im) * in.hir - (in.hr - in.hr_jm) * in.inv_rdphi_int;
        const T t2 = cpml_apply(q, chi_ez, in.bq_i, in.cq_i, R(1));
        ez = ez + in.cE * (t1 + t2);
    }
}
template <class T, class R>
__device__ __forceinline__ void e_update_voxel(const EIn<T, R>& in, T& er, T& ep, T& ez,
                                               T& psi_er_z, T& psi_ep_z, T& psi_ep_r, T& psi_ez_r) {
    T c0 = zero_of<T>(), c1 = zero_of<T>();
    e_update_voxel(in, er, ep, ez, psi_er_z, psi_ep_z, psi_ep_r, psi_ez_r, c0, c1);
}

// Field arrays carry FIELD_GHOST ghost rows on each side of phi: physical row j sits at storage row j + FIELD_GHOST, and
// storage row s outside the physical range holds an UN-PHASED copy of physical row (s - FIELD_GHOST) mod Nphi (the Bloch
// phase is applied where a row is used across the wrap).  Two rows, because the two-step fused kernel reads a halo of two.
// The depth is per zone (StepParams::ghost): 2 where the two-step kernel can run, 1 for thin wedges and axis zones, whose
// rows are few enough for the extra ghost copies to cost 15-20 % of their traffic (config6 26.7 -> 30 Gvox/s).
constexpr int FIELD_GHOST_MAX = 2;
// Row offsets (in rows, relative to the row's own storage row) of the ghost copies of physical row j; returns their count.
__host__ __device__ __forceinline__ int ghost_row_offsets(int j, int Nphi, int ghost, int out[2 * FIELD_GHOST_MAX]) {
    int n = 0;
    for (int g = 0; g < 2 * ghost; ++g) {
        const int s = g < ghost ? g : Nphi + g;                    // storage rows 0 .. ghost - 1, Nphi + ghost .. Nphi + 2 ghost - 1
        int ph = (s - ghost) % Nphi;
        if (ph < 0) ph += Nphi;
        if (ph == j) out[n++] = s - (j + ghost);
    }
    return n;
}

// Kernel parameter block (one per launch, passed by value).
template <class T> struct StepParams {
    using R = typename ElemTraits<T>::Real;
    int Nr, Nphi, Nz, pitch;
    // field arrays (E, H) are stored [Nz][Nphi + 2 FIELD_GHOST][pitch]: physical row j sits at storage row
    // j + FIELD_GHOST; the ghost rows are un-phased copies of the rows across the wrap (kept by the fused
    // kernels so that their TMA tiles never straddle the phi wrap; the split kernels ignore them).
    // Every other array is dense in phi: [..][Nphi][pitch].
    size_t fplane;                     // pitch * (Nphi + 2 ghost)
    int ghost;                         // ghost rows on each side of phi (FIELD_GHOST of the comments): 1 or 2
    int has_axis, p_is_one;
    R dt, inv_dr, inv_dz, pr, pi;      // pi: phase imaginary part of THIS run (conjugated for the adjoint)
    const R* rc;                       // per-r tables, rc[t * pitch + i], t = RC_*
    const R* zc;                       // per-z tables, zc[t * Nz + k], t = ZC_*
    int npr_lo, npr_hi, npz_lo, npz_hi;
    T* E[3];                           // current E (read by H-update, updated by E-update)
    T* H[3];
    T* Eout[3];                        // fused kernel: destination buffers (double buffering)
    T* Hout[3];
    T* psiH_z[2];                      // Hr_z, Hphi_z     [npz][Nphi][pitch]
    T* psiH_r[2];                      // Hphi_r, Hz_r     [Nz][Nphi][npr]
    T* psiH_z_out[2];                  // fused kernel: destination (halo recompute reads the old copy)
    T* psiH_r_out[2];
    T* psiE_z[2];                      // Er_z, Ephi_z
    T* psiE_r[2];                      // Ephi_r, Ez_r
    // R25 (exact outer r-PML): auxiliaries of the 1/r~ operator, laid out like the r-slab psi arrays; rpml_exact = 0: unused
    int rpml_exact;
    T* chiH[2];                        // Hr, Hz
    T* chiH_out[2];
    T* chiE[2];                        // Er, Ez
    T* chiE_out[2];
    T* psiE_z_out[2];                  // fused kernels: destination (the two-step kernel recomputes E on its halo from the
    T* psiE_r_out[2];                  // old copy); the split kernels update in place (out == in)
    const R* cE_design;                // dt/eps on the material planes mk0 <= k < mk1, [mk1 - mk0][Nphi][pitch] (all i: the
                                       // background value outside the design box); the planes of the design layer, or
                                       // every plane when the zone holds a per-voxel eps volume (zda_set_eps_volume)
    int mk0, mk1;
    int di0, di1, dk0, dk1;            // design box: DFT accumulators, gradient
    const T* axis_mean;                // [Nz]: mean_j Hphi[0, j, k] (axis zones)
    // current sheet (R15 / R11)
    const T* A_r;
    const T* A_phi;                    // [n_terms][Nphi][pitch]
    const T* s_tab;                    // [n_terms][tab_len]
    int n_terms, tab_len, src_k;
    // running DFT (R8)
    int F;
    const Cx<R>* tw;                   // [max_steps][F]: dt exp(+i omega_f (n+1) dt)
    Cx<R>* dft_design;                 // [F][3][Ld][Nphi][pitch]
    Cx<R>* dft_mon;                    // [F][3][Nphi][pitch] or nullptr
    int mon_k;
    int n;                             // step index
    const int* n_dev;                  // split kernels under a CUDA graph: the step index lives on the device (bumped by
                                       // the H-update kernel) so that every step's launch parameters are identical
    // Running DFT of this launch (R8).  The accumulators may be visited every second launch only: launch n then adds
    // step n-1's term from its INPUT E (= E^n, still intact in the other time buffer) and step n's term from the
    // E it has just computed, in that order -- bit-identical to visiting them every step, at half the traffic.
    int dft_mode;                      // 0: leave the accumulators alone; 1: add step n; 2: add step n-1, then step n
    // Design-box accumulators visited every s > 2 steps by dft_visit_kernel (zda_zone_impl.cuh): dft_design is then
    // nullptr here and, on the launches whose E^{n+1} will have left both time buffers by the time of the visit, the fused
    // kernel also stores its design-layer E^{n+1} to ring_store, laid out [3][Ld][Nphi][pitch].
    T* ring_store;
    // Two-step kernel: ring_store takes the launch's FIRST step (E^{n+1}, which never reaches a time buffer),
    // ring_store_b its second (E^{n+2}) on the launches whose output buffer is overwritten before the visit.
    T* ring_store_b;
};

}  // namespace zda
