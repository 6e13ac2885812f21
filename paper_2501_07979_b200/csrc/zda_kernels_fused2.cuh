// Two time steps per HBM pass (north_star "temporal blocking (several time steps per HBM pass)").
//
// One launch advances the zone from (E^n, H^{n-1/2}) to (E^{n+2}, H^{n+3/2}): every field is read ONCE and written ONCE per
// TWO steps.  A CTA owns a tile of (r, phi), loads it with a halo of two cells (TMA, as in the one-step kernel), and marches
// along z with step B trailing step A by one plane:
//
//   phase 1   H_A(k)    = H^{n+1/2}(k)   from E^n(k), E^n(k+1), H^{n-1/2}(k)           tile rows 0 .. TJ+2
//   phase 2   E_A(k)    = E^{n+1}(k)     from H_A(k), H_A(k-1), E^n(k)                 tile rows 1 .. TJ+2
//   phase 3   H_B(k-1)  = H^{n+3/2}(k-1) from E_A(k-1), E_A(k), H_A(k-1)               tile rows 1 .. TJ+1
//   phase 4   E_B(k-1)  = E^{n+2}(k-1)   from H_B(k-1), H_B(k-2), E_A(k-1)             tile rows 2 .. TJ+1 (the CTA's own)
//
// Step A is recomputed on a ring one cell wider than step B needs (halo recompute instead of an exchange): in phi by the
// extra warps (rows 0, 1 and TJ+2 are halo rows), in r inside the 32 lanes of a row (lanes LO .. 30 own their 16 bytes,
// lane 0/LO-1 and lane 31 are halo lanes), in z by the chunk's first three planes.  Every halo value is computed from the
// launch's INPUT buffers with the same expressions as its owner (h_update_voxel / e_update_voxel), so the result is
// bit-identical to two single steps; that is why fields and ALL CPML auxiliaries are double-buffered.
// Neighbours: z from registers (the previous plane), r from warp shuffles, phi from small shared-memory row arrays; two
// __syncthreads per plane pair.  The running DFT adds both steps' terms in step order from registers.
#pragma once
#include "zda_kernels_fused.cuh"

namespace zda {

template <int TJ> struct alignas(1024) Fused2Smem {
    static constexpr int ROWS = TJ + 4;                      // tile rows incl. two halo rows on each side
    struct alignas(128) Slot { unsigned char c[3][ROWS][FUSED_ROW_BYTES]; };
    Slot E[3];                                               // E^n planes k, k+1, k+2
    Slot H[2];                                               // H^{n-1/2} planes k, k+1
    alignas(16) unsigned char HnA[2][TJ + 3][FUSED_PAY_BYTES];     // step A: new {Hr, Hz} of rows 0..TJ+2
    alignas(16) unsigned char EA[2][2][TJ + 3][FUSED_PAY_BYTES];   // step A: new {Er, Ez} of rows 1..TJ+2, double-buffered over k
    alignas(16) unsigned char HnB[2][TJ + 2][FUSED_PAY_BYTES];     // step B: new {Hr, Hz} of rows 1..TJ+1
    alignas(16) unsigned char coef[12][FUSED_PAY_BYTES];           // per-r tables of the tile's 32 units
    unsigned long long barE[3], barH[2];
};

__device__ __forceinline__ float shfl_down1(float x) { return __shfl_down_sync(0xffffffffu, x, 1); }
__device__ __forceinline__ double shfl_down1(double x) { return __shfl_down_sync(0xffffffffu, x, 1); }
template <class R> __device__ __forceinline__ Cx<R> shfl_down1(Cx<R> x) { return {shfl_down1(x.x), shfl_down1(x.y)}; }

template <class T, int TJ, bool RS>
__device__ __forceinline__ void fused2_body(const StepParams<T>& P, const CUtensorMap& tmap, const FusedGeom& G) {
    using R = typename ElemTraits<T>::Real;
    using V = VecT<T>;
    using Smem = Fused2Smem<TJ>;
    constexpr int VEC = V::N;
    constexpr int W = (int)sizeof(T) / 4;
    constexpr int NW = TJ + 3;                          // warps: one per tile row 0 .. TJ+2
    constexpr int LO = (2 + VEC - 1) / VEC;             // first owning lane: two halo cells on the low side
    constexpr int NU_OUT = 31 - LO;                     // owning lanes LO .. 30 (lane 31's last cell is a halo cell)
    constexpr int TI_OUT = NU_OUT * VEC;
    constexpr unsigned SLOT_BYTES = 3u * (TJ + 4) * FUSED_ROW_BYTES;

    extern __shared__ unsigned char smem_raw[];
    Smem& S = *reinterpret_cast<Smem*>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u));

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int b = blockIdx.x;
    const int crank = b % G.cluster; b /= G.cluster;
    const int ti = b % G.n_ti; b /= G.n_ti;
    const int tj = (b % G.n_tjc) * G.cluster + crank;
    const int zc = b / G.n_tjc;
    const bool tile_ok = tj < G.n_tj;
    const int a0 = ti * TI_OUT - LO * VEC;              // cell index of lane 0's first element
    const int j0 = tj * TJ;
    const int Nr = P.Nr, Nphi = P.Nphi, Nz = P.Nz, pitch = P.pitch;
    const int ka = zc * G.chunk, kb = min(ka + G.chunk, Nz);
    const int kEA0 = ka > 0 ? ka - 1 : 0;               // first plane of E_A / H_B
    const int kstart = ka > 1 ? ka - 2 : 0;             // first plane of H_A
    const int nit = kb - kstart + 1;                    // iteration it: step A on plane kstart + it, step B one below
    const int nE = min(kb + 1, Nz) - kstart + 1;        // E^n planes kstart .. min(kb + 1, Nz) (plane Nz is the zero ghost)
    const int nH = min(kb, Nz - 1) - kstart + 1;        // H^{n-1/2} planes kstart .. min(kb, Nz - 1)
    const size_t row = (size_t)pitch, plane = row * Nphi, fplane = P.fplane;
    const int npr = P.npr_lo + P.npr_hi;

    auto issueE = [&](int e) __attribute__((always_inline)) {
        unsigned long long* bar = &S.barE[e % 3];
        mbar_expect_tx(bar, SLOT_BYTES);
        tma_load_4d(&S.E[e % 3], &tmap, bar, a0 * W, j0, kstart + e, G.aE);
    };
    auto issueH = [&](int h) __attribute__((always_inline)) {
        unsigned long long* bar = &S.barH[h & 1];
        mbar_expect_tx(bar, SLOT_BYTES);
        tma_load_4d(&S.H[h & 1], &tmap, bar, a0 * W, j0, kstart + h, G.aH);
    };

    if (tid == 0) {
        for (int s = 0; s < 3; ++s) mbar_init(&S.barE[s], 1);
        for (int s = 0; s < 2; ++s) mbar_init(&S.barH[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int e = 0; e < 3 && e < nE; ++e) issueE(e);
        for (int h = 0; h < 2 && h < nH; ++h) issueH(h);
    }
    {
        constexpr int tabs[12] = {RC_INV_RDPHI_INT, RC_INV_RDPHI_HALF, RC_CA, RC_CB, RC_CC, RC_CD,
                                  RC_B_H, RC_C_H, RC_IK_H, RC_B_I, RC_C_I, RC_IK_I};
        for (int t = tid; t < (RS ? 12 : 6) * 32 * VEC; t += NW * 32) {
            const int w = t / (32 * VEC), x = t % (32 * VEC), idx = a0 + x;
            reinterpret_cast<R*>(S.coef[w])[x] = (idx >= 0 && idx < pitch) ? P.rc[tabs[w] * pitch + idx] : R(0);
        }
    }
    __syncthreads();

    // ---- per-thread constants ---------------------------------------------------------------
    const int y = warp;                                  // tile row; physical row j0 - 2 + y
    const int jraw = j0 - 2 + y;
    int jm = jraw % Nphi; if (jm < 0) jm += Nphi;
    const int j = jm;                                    // physical row (halo rows wrap, several times when Nphi is tiny)
    const bool rowHA = tile_ok && (jraw <= Nphi);                              // H_A: rows -2 .. Nphi
    const bool rowEA = rowHA && (y >= 1);                                      // E_A: rows -1 .. Nphi
    const bool rowHB = tile_ok && (y >= 1) && (y <= TJ + 1) && (jraw <= Nphi - 1);   // H_B: rows -1 .. Nphi - 1
    const bool own = rowHB && (y >= 2);                                        // E_B and the stores: the tile's own rows
    const bool j_last = (j == Nphi - 1), j_first = (j == 0);
    const int ig = a0 + lane * VEC;
    const bool col_ok = (ig >= 0) && (ig < pitch);       // pitch % 32 == 0: a group is all inside or all outside
    const bool out_lane = (lane >= LO) && (lane < 31) && (ig < Nr);

    struct alignas(VEC * sizeof(R)) CoefV { R v[VEC]; };
    auto coefv = [&](int w) __attribute__((always_inline)) { return reinterpret_cast<const CoefV*>(S.coef[w])[lane]; };
    int ir[VEC];
    bool any_rs = false, in_dom[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
        const int idx = ig + e;
        in_dom[e] = (idx >= 0) && (idx < Nr);
        ir[e] = (RS && in_dom[e]) ? slab_index(idx, Nr, P.npr_lo, P.npr_hi) : -1;
        any_rs = any_rs || (ir[e] >= 0);
    }

    const size_t pj = (size_t)j * row + (size_t)(col_ok ? ig : 0);     // (j, ig) in the dense [Nphi][pitch] arrays
    size_t foB = (size_t)(kstart - 1) * fplane + (size_t)(j + FIELD_GHOST_MAX) * row + (size_t)(col_ok ? ig : 0);   // step B plane
    int gro[2 * FIELD_GHOST_MAX];
    const int n_gh = ghost_row_offsets(j, Nphi, FIELD_GHOST_MAX, gro);
    const int g_off0 = n_gh > 0 ? gro[0] * pitch : 0;     // in elements: at most (Nphi + 2) pitch < 2^31; further copies
                                                         // (tiny Nphi only) behind a rare branch
    const size_t orr_step = (size_t)Nphi * npr;
    size_t orrA = ((size_t)kstart * Nphi + j) * npr;     // (kA, j, 0) in the r-slab psi arrays

    // ---- state carried from one plane to the next ----------------------------------------------
    V hAp[3], eAp[3];                  // H_A, E_A of the previous plane (= step B's plane)
    T hBr_km[VEC], hBp_km[VEC];        // H_B {r, phi} two planes down (z-neighbour of E_B)
    V pzHp[2], pzEp[2];                // z-slab psi after step A, previous plane
    T prHp[2][VEC], prEp[2][VEC];      // r-slab psi after step A, previous plane
    R cEp[VEC];                        // dt/eps of the previous plane
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int e = 0; e < VEC; ++e) { hAp[c].v[e] = zero_of<T>(); eAp[c].v[e] = zero_of<T>(); }
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
        hBr_km[e] = hBp_km[e] = zero_of<T>();
        cEp[e] = R(0);
#pragma unroll
        for (int c = 0; c < 2; ++c) { pzHp[c].v[e] = pzEp[c].v[e] = zero_of<T>(); prHp[c][e] = prEp[c][e] = zero_of<T>(); }
    }

    auto plane_iter = [&](auto zs_tag, auto lean_tag, const int it) __attribute__((always_inline)) {
        constexpr bool zs = decltype(zs_tag)::value;     // plane kA or plane kB lies in a z-slab
        // lean: an interior plane pair with nothing special on it -- all four phases run, neither plane is a material,
        // design, source or monitor plane (next_special below) -- so every per-plane predicate is a compile-time constant
        // and the code behind it is gone; the arithmetic that remains is the full body's, instruction for instruction
        constexpr bool lean = decltype(lean_tag)::value;
        static_assert(!(zs && lean), "the lean body has no z-slab code");
        const int kA = kstart + it, kB = kA - 1;
        const bool doHA = lean || kA < Nz;               // the last chunk's last iteration has kA == Nz: E_A there is the zero ghost
        const bool doEA = lean || (doHA && kA >= kEA0);
        const bool doHB = lean || kB >= kEA0;
        const bool doEB = lean || kB >= ka;
        const int kzA = (zs && doHA) ? slab_index(kA, Nz, P.npz_lo, P.npz_hi) : -1;
        const int kzB = (zs && kB >= 0) ? slab_index(kB, Nz, P.npz_lo, P.npz_hi) : -1;
        const bool kmA = !lean && doHA && (kA >= P.mk0 && kA < P.mk1);
        const bool kdB = !lean && (kB >= P.dk0 && kB < P.dk1);
        const size_t ozA = (size_t)(kzA >= 0 ? kzA : 0) * plane + pj;
        const size_t ozB = (size_t)(kzB >= 0 ? kzB : 0) * plane + pj;

        // ---- global operands of step A's plane, requested before the tile wait -------------------
        V pzH[2], pzE[2];
        T prH[2][VEC], prE[2][VEC];
        R cEv[VEC];
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            cEv[e] = R(0);
#pragma unroll
            for (int c = 0; c < 2; ++c) { pzH[c].v[e] = pzE[c].v[e] = zero_of<T>(); prH[c][e] = prE[c][e] = zero_of<T>(); }
        }
        if (zs && kzA >= 0 && rowHA && col_ok) {
            pzH[0] = ldg_early(reinterpret_cast<const V*>(P.psiH_z[0] + ozA));
            pzH[1] = ldg_early(reinterpret_cast<const V*>(P.psiH_z[1] + ozA));
            if (rowEA && doEA) {
                pzE[0] = ldg_early(reinterpret_cast<const V*>(P.psiE_z[0] + ozA));
                pzE[1] = ldg_early(reinterpret_cast<const V*>(P.psiE_z[1] + ozA));
            }
        }
        if (RS && any_rs && rowHA && doHA) {
#pragma unroll
            for (int e = 0; e < VEC; ++e)
                if (ir[e] >= 0) {
                    prH[0][e] = ldg_early(P.psiH_r[0] + orrA + ir[e]); prH[1][e] = ldg_early(P.psiH_r[1] + orrA + ir[e]);
                    if (rowEA && doEA) {
                        prE[0][e] = ldg_early(P.psiE_r[0] + orrA + ir[e]); prE[1][e] = ldg_early(P.psiE_r[1] + orrA + ir[e]);
                    }
                }
        }
        if (kmA && rowEA && doEA && col_ok) {
            struct alignas(VEC * sizeof(R)) CEV { R v[VEC]; };
            const CEV c = ldg_early(reinterpret_cast<const CEV*>(P.cE_design + (size_t)(kA - P.mk0) * plane + pj));
#pragma unroll
            for (int e = 0; e < VEC; ++e) cEv[e] = c.v[e];
        }
        const bool monB = !lean && (kB == P.mon_k) && (P.dft_mon != nullptr);
        const bool dboxB = kdB && (ig < P.di1) && (ig + VEC > P.di0);
        const bool dgrpB = dboxB && (P.dft_design != nullptr);
        if (own && doEB && out_lane) {
            if (dgrpB) {
                const int Ld = P.dk1 - P.dk0;
                for (int fc = 0; fc < 3 * P.F; ++fc)
                    prefetch_l2(P.dft_design + ((size_t)fc * Ld + (kB - P.dk0)) * plane + pj);
            }
            if (monB)
                for (int fc = 0; fc < 3 * P.F; ++fc) prefetch_l2(P.dft_mon + (size_t)fc * plane + pj);
        }
        // per-plane scalars
        const R cbgA = doHA ? ldg_early(P.zc + ZC_CE_BG * Nz + kA) : R(0);
        R bzHA = R(0), czHA = R(0), ikzHA = R(1), bzEA = R(0), czEA = R(0), ikzEA = R(1);
        R bzHB = R(0), czHB = R(0), ikzHB = R(1), bzEB = R(0), czEB = R(0), ikzEB = R(1);
        if (zs) {
            if (kzA >= 0) {
                bzHA = ldg_early(P.zc + ZC_B_H * Nz + kA); czHA = ldg_early(P.zc + ZC_C_H * Nz + kA); ikzHA = ldg_early(P.zc + ZC_IK_H * Nz + kA);
                bzEA = ldg_early(P.zc + ZC_B_I * Nz + kA); czEA = ldg_early(P.zc + ZC_C_I * Nz + kA); ikzEA = ldg_early(P.zc + ZC_IK_I * Nz + kA);
            }
            if (kzB >= 0) {
                bzHB = ldg_early(P.zc + ZC_B_H * Nz + kB); czHB = ldg_early(P.zc + ZC_C_H * Nz + kB); ikzHB = ldg_early(P.zc + ZC_IK_H * Nz + kB);
                bzEB = ldg_early(P.zc + ZC_B_I * Nz + kB); czEB = ldg_early(P.zc + ZC_C_I * Nz + kB); ikzEB = ldg_early(P.zc + ZC_IK_I * Nz + kB);
            }
        }
        // step B's r-neighbours of E_A(kB): from the previous iteration's registers, requested before the tile wait
        T epB_nx = shfl_down1(eAp[1].v[0]), ezB_nx = shfl_down1(eAp[2].v[0]);
        if (lane == 31) { epB_nx = zero_of<T>(); ezB_nx = zero_of<T>(); }     // halo cell: H_B is not valid there
        if (G.cluster > 1 && it > 0) cluster_wait();
        if (doHA) {
            if (it == 0) mbar_wait(&S.barE[0], 0);
            mbar_wait(&S.barE[(it + 1) % 3], ((it + 1) / 3) & 1);
            mbar_wait(&S.barH[it & 1], (it >> 1) & 1);
        }
        const typename Smem::Slot& Ek = S.E[it % 3];
        const typename Smem::Slot& Ek1 = S.E[(it + 1) % 3];
        const typename Smem::Slot& Hk = S.H[it & 1];
        const int buf = it & 1;

        // ================= phase 1: H_A(kA), rows 0 .. TJ+2 =================
        V eN[3], hA[3];
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int e = 0; e < VEC; ++e) { eN[c].v[e] = zero_of<T>(); hA[c].v[e] = zero_of<T>(); }
        if (rowHA && doHA) {
            eN[0] = lds_vec<T>(Ek.c[0][y], lane);
            eN[1] = lds_vec<T>(Ek.c[1][y], lane);
            eN[2] = lds_vec<T>(Ek.c[2][y], lane);
            const T ep_nx = lds_elem<T>(Ek.c[1][y], lane + 1, 0);
            const T ez_nx = lds_elem<T>(Ek.c[2][y], lane + 1, 0);
            V er_jp = lds_vec<T>(Ek.c[0][y + 1], lane);
            V ez_jp = lds_vec<T>(Ek.c[2][y + 1], lane);
            if (j_last) {
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    er_jp.v[e] = phase_mul(P.pr, P.pi, er_jp.v[e]);
                    ez_jp.v[e] = phase_mul(P.pr, P.pi, ez_jp.v[e]);
                }
            }
            const V er_kp = lds_vec<T>(Ek1.c[0][y], lane);
            const V ep_kp = lds_vec<T>(Ek1.c[1][y], lane);
            hA[0] = lds_vec<T>(Hk.c[0][y], lane);
            hA[1] = lds_vec<T>(Hk.c[1][y], lane);
            hA[2] = lds_vec<T>(Hk.c[2][y], lane);
            const CoefV c_rI = coefv(0), c_rH = coefv(1), c_ca = coefv(2), c_cb = coefv(3);
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                HIn<T, R> in;
                in.er = eN[0].v[e]; in.ep = eN[1].v[e]; in.ez = eN[2].v[e];
                in.er_jp = er_jp.v[e]; in.ez_jp = ez_jp.v[e];
                in.er_kp = er_kp.v[e]; in.ep_kp = ep_kp.v[e];
                in.ep_ip = (e + 1 < VEC) ? eN[1].v[(e + 1) % VEC] : ep_nx;
                in.ez_ip = (e + 1 < VEC) ? eN[2].v[(e + 1) % VEC] : ez_nx;
                in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.ca = c_ca.v[e]; in.cb = c_cb.v[e];
                in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.dt = P.dt;
                in.bz = bzHA; in.cz = czHA; in.ikz = ikzHA;
                in.zs = zs && (kzA >= 0); in.rs = RS && ir[e] >= 0; in.skip_hr = false;
                in.br = in.cr = R(0); in.ikr = R(1);
                if (RS) { in.br = coefv(6).v[e]; in.cr = coefv(7).v[e]; in.ikr = coefv(8).v[e]; }
                h_update_voxel(in, hA[0].v[e], hA[1].v[e], hA[2].v[e], pzH[0].v[e], pzH[1].v[e], prH[0][e], prH[1][e]);
            }
            *reinterpret_cast<V*>(&S.HnA[0][y][16 * lane]) = hA[0];
            *reinterpret_cast<V*>(&S.HnA[1][y][16 * lane]) = hA[2];
        }
        // r-neighbours of H_A for phase 2, in flight across the barrier
        T hpA_w = shfl_up1(hA[1].v[VEC - 1]), hzA_w = shfl_up1(hA[2].v[VEC - 1]);
        if (lane == 0) { hpA_w = zero_of<T>(); hzA_w = zero_of<T>(); }      // halo cell: E_A is not valid there
        __syncthreads();
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            if (it + 3 < nE) issueE(it + 3);
            if (it + 2 < nH) issueH(it + 2);
        }

        // ================= phase 2: E_A(kA), rows 1 .. TJ+2 =================
        V eA[3];                         // stays zero on the virtual plane kA == Nz: E_A there is the PEC ghost
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int e = 0; e < VEC; ++e) eA[c].v[e] = zero_of<T>();
        R cEA[VEC];
#pragma unroll
        for (int e = 0; e < VEC; ++e) cEA[e] = (kmA && col_ok) ? cEv[e] : cbgA;
        if (rowEA && doEA) {
            V hr_jm = *reinterpret_cast<const V*>(&S.HnA[0][y - 1][16 * lane]);
            V hz_jm = *reinterpret_cast<const V*>(&S.HnA[1][y - 1][16 * lane]);
            if (j_first) {
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    hr_jm.v[e] = phase_mul(P.pr, -P.pi, hr_jm.v[e]);
                    hz_jm.v[e] = phase_mul(P.pr, -P.pi, hz_jm.v[e]);
                }
            }
            const T hp_w = hpA_w, hz_w = hzA_w;
            T jr[VEC], jp[VEC];
#pragma unroll
            for (int e = 0; e < VEC; ++e) { jr[e] = zero_of<T>(); jp[e] = zero_of<T>(); }
            if (!lean && kA == P.src_k && P.n_terms > 0 && P.n < P.tab_len && col_ok) {
                for (int q = 0; q < P.n_terms; ++q) {
                    const T s = P.s_tab[(size_t)q * P.tab_len + P.n];
                    const V ar = ldg_vec(P.A_r + (size_t)q * plane + pj), ap = ldg_vec(P.A_phi + (size_t)q * plane + pj);
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        if constexpr (ElemTraits<T>::cplx) { jr[e] = jr[e] + cmul(s, ar.v[e]); jp[e] = jp[e] + cmul(s, ap.v[e]); }
                        else { jr[e] = jr[e] + s * ar.v[e]; jp[e] = jp[e] + s * ap.v[e]; }
                    }
                }
            }
            eA[0] = eN[0]; eA[1] = eN[1]; eA[2] = eN[2];
            const CoefV c_rI = coefv(0), c_rH = coefv(1), c_cc = coefv(4), c_cd = coefv(5);
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                EIn<T, R> in;
                in.hr = hA[0].v[e]; in.hp = hA[1].v[e]; in.hz = hA[2].v[e];
                in.hr_jm = hr_jm.v[e]; in.hz_jm = hz_jm.v[e];
                in.hr_km = hAp[0].v[e]; in.hp_km = hAp[1].v[e];
                in.hp_im = (e > 0) ? hA[1].v[(e + VEC - 1) % VEC] : hp_w;
                in.hz_im = (e > 0) ? hA[2].v[(e + VEC - 1) % VEC] : hz_w;
                in.jr = jr[e]; in.jp = jp[e];
                in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.cc = c_cc.v[e]; in.cd = c_cd.v[e];
                in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.cE = cEA[e];
                in.bz = bzEA; in.cz = czEA; in.ikz = ikzEA;
                in.zs = zs && (kzA >= 0); in.rs = RS && ir[e] >= 0;
                in.k_pos = zs ? (kA > 0) : true;         // plane 0 is always handled by a z-slab body (it_a below)
                in.i_pos = RS ? (ig + e > 0) : true;     // interior tiles have no i = 0 column
                in.br = in.cr = R(0); in.ikr = R(1);
                if (RS) { in.br = coefv(9).v[e]; in.cr = coefv(10).v[e]; in.ikr = coefv(11).v[e]; }
                e_update_voxel(in, eA[0].v[e], eA[1].v[e], eA[2].v[e], pzE[0].v[e], pzE[1].v[e], prE[0][e], prE[1][e]);
                if (RS && !in_dom[e]) { eA[0].v[e] = zero_of<T>(); eA[1].v[e] = zero_of<T>(); eA[2].v[e] = zero_of<T>(); }   // PEC ghost
            }
            *reinterpret_cast<V*>(&S.EA[buf][0][y][16 * lane]) = eA[0];
            *reinterpret_cast<V*>(&S.EA[buf][1][y][16 * lane]) = eA[2];
        }

        // ================= phase 3: H_B(kB), rows 1 .. TJ+1 =================
        V hB[3];
        hB[0] = hAp[0]; hB[1] = hAp[1]; hB[2] = hAp[2];
        V pzHB[2];
        T prHB[2][VEC];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                pzHB[c].v[e] = zs ? pzHp[c].v[e] : zero_of<T>();      // bodies without a slab carry no psi state
                prHB[c][e] = RS ? prHp[c][e] : zero_of<T>();
            }
        }
        if (rowHB && doHB) {
            V er_jp = *reinterpret_cast<const V*>(&S.EA[buf ^ 1][0][y + 1][16 * lane]);
            V ez_jp = *reinterpret_cast<const V*>(&S.EA[buf ^ 1][1][y + 1][16 * lane]);
            if (j_last) {
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    er_jp.v[e] = phase_mul(P.pr, P.pi, er_jp.v[e]);
                    ez_jp.v[e] = phase_mul(P.pr, P.pi, ez_jp.v[e]);
                }
            }
            const T ep_nx = epB_nx, ez_nx = ezB_nx;
            const CoefV c_rI = coefv(0), c_rH = coefv(1), c_ca = coefv(2), c_cb = coefv(3);
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                HIn<T, R> in;
                in.er = eAp[0].v[e]; in.ep = eAp[1].v[e]; in.ez = eAp[2].v[e];
                in.er_jp = er_jp.v[e]; in.ez_jp = ez_jp.v[e];
                in.er_kp = eA[0].v[e]; in.ep_kp = eA[1].v[e];
                in.ep_ip = (e + 1 < VEC) ? eAp[1].v[(e + 1) % VEC] : ep_nx;
                in.ez_ip = (e + 1 < VEC) ? eAp[2].v[(e + 1) % VEC] : ez_nx;
                in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.ca = c_ca.v[e]; in.cb = c_cb.v[e];
                in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.dt = P.dt;
                in.bz = bzHB; in.cz = czHB; in.ikz = ikzHB;
                in.zs = zs && (kzB >= 0); in.rs = RS && ir[e] >= 0; in.skip_hr = false;
                in.br = in.cr = R(0); in.ikr = R(1);
                if (RS) { in.br = coefv(6).v[e]; in.cr = coefv(7).v[e]; in.ikr = coefv(8).v[e]; }
                h_update_voxel(in, hB[0].v[e], hB[1].v[e], hB[2].v[e], pzHB[0].v[e], pzHB[1].v[e], prHB[0][e], prHB[1][e]);
            }
            *reinterpret_cast<V*>(&S.HnB[0][y][16 * lane]) = hB[0];
            *reinterpret_cast<V*>(&S.HnB[1][y][16 * lane]) = hB[2];
            // the new H leaves for HBM here, ahead of the barrier: its registers stay live (phase 4, next plane's z-neighbour),
            // so these stores hold nothing up, and they drain while the warps meet
            if (own && doEB && out_lane) {
                stg_vec(P.Hout[0] + foB, hB[0]); stg_vec(P.Hout[1] + foB, hB[1]); stg_vec(P.Hout[2] + foB, hB[2]);
            }
        }
        T hpB_w = shfl_up1(hB[1].v[VEC - 1]), hzB_w = shfl_up1(hB[2].v[VEC - 1]);   // r-neighbours of H_B for phase 4
        if (lane == 0) { hpB_w = zero_of<T>(); hzB_w = zero_of<T>(); }
        __syncthreads();

        // ================= phase 4: E_B(kB), own rows; stores =================
        if (own && doEB) {
            V hr_jm = *reinterpret_cast<const V*>(&S.HnB[0][y - 1][16 * lane]);
            V hz_jm = *reinterpret_cast<const V*>(&S.HnB[1][y - 1][16 * lane]);
            if (j_first) {
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    hr_jm.v[e] = phase_mul(P.pr, -P.pi, hr_jm.v[e]);
                    hz_jm.v[e] = phase_mul(P.pr, -P.pi, hz_jm.v[e]);
                }
            }
            const T hp_w = hpB_w, hz_w = hzB_w;
            T jr[VEC], jp[VEC];
#pragma unroll
            for (int e = 0; e < VEC; ++e) { jr[e] = zero_of<T>(); jp[e] = zero_of<T>(); }
            if (!lean && kB == P.src_k && P.n_terms > 0 && P.n + 1 < P.tab_len && col_ok) {
                for (int q = 0; q < P.n_terms; ++q) {
                    const T s = P.s_tab[(size_t)q * P.tab_len + P.n + 1];
                    const V ar = ldg_vec(P.A_r + (size_t)q * plane + pj), ap = ldg_vec(P.A_phi + (size_t)q * plane + pj);
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        if constexpr (ElemTraits<T>::cplx) { jr[e] = jr[e] + cmul(s, ar.v[e]); jp[e] = jp[e] + cmul(s, ap.v[e]); }
                        else { jr[e] = jr[e] + s * ar.v[e]; jp[e] = jp[e] + s * ap.v[e]; }
                    }
                }
            }
            V eB[3];
            eB[0] = eAp[0]; eB[1] = eAp[1]; eB[2] = eAp[2];
            V pzEB[2];
            T prEB[2][VEC];
#pragma unroll
            for (int c = 0; c < 2; ++c) {
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    pzEB[c].v[e] = zs ? pzEp[c].v[e] : zero_of<T>();
                    prEB[c][e] = RS ? prEp[c][e] : zero_of<T>();
                }
            }
            const CoefV c_rI = coefv(0), c_rH = coefv(1), c_cc = coefv(4), c_cd = coefv(5);
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                EIn<T, R> in;
                in.hr = hB[0].v[e]; in.hp = hB[1].v[e]; in.hz = hB[2].v[e];
                in.hr_jm = hr_jm.v[e]; in.hz_jm = hz_jm.v[e];
                in.hr_km = hBr_km[e]; in.hp_km = hBp_km[e];
                in.hp_im = (e > 0) ? hB[1].v[(e + VEC - 1) % VEC] : hp_w;
                in.hz_im = (e > 0) ? hB[2].v[(e + VEC - 1) % VEC] : hz_w;
                in.jr = jr[e]; in.jp = jp[e];
                in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.cc = c_cc.v[e]; in.cd = c_cd.v[e];
                in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.cE = cEp[e];
                in.bz = bzEB; in.cz = czEB; in.ikz = ikzEB;
                in.zs = zs && (kzB >= 0); in.rs = RS && ir[e] >= 0;
                in.k_pos = zs ? (kB > 0) : true; in.i_pos = RS ? (ig + e > 0) : true;
                in.br = in.cr = R(0); in.ikr = R(1);
                if (RS) { in.br = coefv(9).v[e]; in.cr = coefv(10).v[e]; in.ikr = coefv(11).v[e]; }
                e_update_voxel(in, eB[0].v[e], eB[1].v[e], eB[2].v[e], pzEB[0].v[e], pzEB[1].v[e], prEB[0][e], prEB[1][e]);
            }
            if (out_lane) {
                stg_vec(P.Eout[0] + foB, eB[0]); stg_vec(P.Eout[1] + foB, eB[1]); stg_vec(P.Eout[2] + foB, eB[2]);
                if (n_gh > 0) {
                    for (int g = 0; g < n_gh; ++g) {
                        const ptrdiff_t o = g == 0 ? (ptrdiff_t)g_off0 : (ptrdiff_t)gro[g] * (ptrdiff_t)row;
                        stg_vec(P.Hout[0] + foB + o, hB[0]); stg_vec(P.Hout[1] + foB + o, hB[1]); stg_vec(P.Hout[2] + foB + o, hB[2]);
                        stg_vec(P.Eout[0] + foB + o, eB[0]); stg_vec(P.Eout[1] + foB + o, eB[1]); stg_vec(P.Eout[2] + foB + o, eB[2]);
                    }
                }
                if (zs && kzB >= 0) {
                    stg_vec(P.psiH_z_out[0] + ozB, pzHB[0]); stg_vec(P.psiH_z_out[1] + ozB, pzHB[1]);
                    stg_vec(P.psiE_z_out[0] + ozB, pzEB[0]); stg_vec(P.psiE_z_out[1] + ozB, pzEB[1]);
                }
                if (RS && any_rs) {
                    const size_t orrB = orrA - orr_step;
#pragma unroll
                    for (int e = 0; e < VEC; ++e)
                        if (ir[e] >= 0) {
                            P.psiH_r_out[0][orrB + ir[e]] = prHB[0][e]; P.psiH_r_out[1][orrB + ir[e]] = prHB[1][e];
                            P.psiE_r_out[0][orrB + ir[e]] = prEB[0][e]; P.psiE_r_out[1][orrB + ir[e]] = prEB[1][e];
                        }
                }
                if (dboxB && P.ring_store != nullptr) {       // step A's design-layer E for a later accumulator visit
                    const size_t Lp = (size_t)(P.dk1 - P.dk0) * plane;
                    T* rp = P.ring_store + (size_t)(kB - P.dk0) * plane + pj;
                    stg_vec(rp, eAp[0]); stg_vec(rp + Lp, eAp[1]); stg_vec(rp + 2 * Lp, eAp[2]);
                }
                if (dboxB && P.ring_store_b != nullptr) {     // step B's
                    const size_t Lp = (size_t)(P.dk1 - P.dk0) * plane;
                    T* rp = P.ring_store_b + (size_t)(kB - P.dk0) * plane + pj;
                    stg_vec(rp, eB[0]); stg_vec(rp + Lp, eB[1]); stg_vec(rp + 2 * Lp, eB[2]);
                }
                // running DFT (R8): step n's term (E_A), then step n+1's (E_B), in that order
                if (dgrpB || monB) {
                    const int Ld = P.dk1 - P.dk0;
                    for (int f = 0; f < P.F; ++f) {
                        const Cx<R> twA = P.tw[(size_t)P.n * P.F + f];
                        const Cx<R> twB = P.tw[(size_t)(P.n + 1) * P.F + f];
                        if (dgrpB)
                            dft_accumulate<T, R, VEC>(P.dft_design + ((size_t)f * 3 * Ld + (kB - P.dk0)) * plane + pj,
                                                      (size_t)Ld * plane, twA, eAp[0], eAp[1], eAp[2], twB, eB[0], eB[1], eB[2]);
                        if (monB)
                            dft_accumulate<T, R, VEC>(P.dft_mon + (size_t)f * 3 * plane + pj, plane, twA, eAp[0], eAp[1], eAp[2],
                                                      twB, eB[0], eB[1], eB[2]);
                    }
                }
            }
        }
        if (rowHB && doHB) {
#pragma unroll
            for (int e = 0; e < VEC; ++e) { hBr_km[e] = hB[0].v[e]; hBp_km[e] = hB[1].v[e]; }
        }
        // ---- rotate: this plane's step-A results become the next iteration's step-B inputs ----------
#pragma unroll
        for (int c = 0; c < 3; ++c) { hAp[c] = hA[c]; eAp[c] = eA[c]; }
#pragma unroll
        for (int c = 0; c < 2; ++c) {
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                if (zs) { pzHp[c].v[e] = pzH[c].v[e]; pzEp[c].v[e] = pzE[c].v[e]; }
                if (RS) { prHp[c][e] = prH[c][e]; prEp[c][e] = prE[c][e]; }
            }
        }
#pragma unroll
        for (int e = 0; e < VEC; ++e) cEp[e] = cEA[e];
        foB += fplane;
        orrA += orr_step;
        if (G.cluster > 1 && it + 1 < nit) cluster_arrive();
    };
    // three iteration ranges: planes kA or kB in the low z-slab, interior, in the high z-slab
    // kB = kstart + it - 1 < max(npz_lo, 1): the slab planes, and plane 0 (its PEC predicate lives in the slab body only)
    const int it_a = min(max(max(P.npz_lo, 1) + 1 - kstart, 0), nit);
    const int it_b = min(max(Nz - P.npz_hi - kstart, it_a), nit);          // kA = kstart + it < Nz - npz_hi
    // Interior iterations that are special: the chunk's start-up (a phase is still off), kA on a material plane or the
    // source plane, kB on a design-layer, source or monitor plane.  next_special(x) = the first such iteration >= x.
    auto next_special = [&](const int x) __attribute__((always_inline)) {
        int r = it_b;
        auto span = [&](const int lo, const int hi) __attribute__((always_inline)) {     // iterations lo .. hi - 1 are special
            if (lo < hi && hi > x) r = min(r, max(lo, x));
        };
        span(0, ka - kstart + 1);                                   // until kB >= ka every phase has started
        span(P.mk0 - kstart, P.mk1 - kstart);                       // kA in [mk0, mk1)
        span(P.dk0 + 1 - kstart, P.dk1 + 1 - kstart);               // kB in [dk0, dk1)
        span(P.src_k - kstart, P.src_k + 2 - kstart);               // kA or kB == src_k
        span(P.mon_k + 1 - kstart, P.mon_k + 2 - kstart);           // kB == mon_k
        return r;
    };
    int it = 0;
#pragma unroll 1
    for (; it < it_a; ++it) plane_iter(std::true_type{}, std::false_type{}, it);
#pragma unroll 1
    while (it < it_b) {
        const int stop = next_special(it);
        if (stop > it) {
#pragma unroll 1
            for (; it < stop; ++it) plane_iter(std::false_type{}, std::true_type{}, it);
        } else {
            plane_iter(std::false_type{}, std::false_type{}, it);
            ++it;
        }
    }
#pragma unroll 1
    for (; it < nit; ++it) plane_iter(std::true_type{}, std::false_type{}, it);
}

template <class T, int TJ, int MINB>
__global__ void __launch_bounds__((TJ + 3) * 32, MINB)
fused2_step_kernel(const __grid_constant__ StepParams<T> P, const __grid_constant__ CUtensorMap tmap, const FusedGeom G) {
    constexpr int VEC = VecT<T>::N;
    constexpr int LO = (2 + VEC - 1) / VEC;
    constexpr int TI_OUT = (31 - LO) * VEC;
    const int a0 = (((int)blockIdx.x / G.cluster) % G.n_ti) * TI_OUT - LO * VEC;
    // CTA-uniform: the tile touches an r-CPML slab or the radial ends of the grid (PEC predicates, cells outside [0, Nr))
    const bool tile_rs = (a0 < P.npr_lo) || (a0 + 32 * VEC > P.Nr - P.npr_hi) || (a0 <= 0) || (a0 + 32 * VEC > P.Nr);
    if (tile_rs) fused2_body<T, TJ, true>(P, tmap, G);
    else fused2_body<T, TJ, false>(P, tmap, G);
}

// ---- host side -------------------------------------------------------------------------------------
template <class R> struct Fused2Plan {
    CUtensorMap tmap;
    FusedGeom G;
    int tj = 5, minb = 2;
    size_t smem_bytes = 0;
    std::string nm;
    bool attr_done[2] = {false, false};

    static bool supported(const zda_zone_desc& d) { return !d.has_axis && field_ghost(d) == 2; }   // needs the two-row halo
    static int choose_tj(int Nphi, int opt_tj) {
        if (opt_tj == 5 || opt_tj == 9 || opt_tj == 13) return opt_tj;
        // measured on config4 / config3 (Gvox/s): 4 rows x 2 CTAs/SM 65, 5 x 2 73 / 40, 5 x 1 (255 registers) 76, 7 x 1 82,
        // 9 x 1 93 / 52, 13 x 1 89 (profiles/r02_fused2.md)
        return Nphi >= 9 ? 9 : 5;
    }
    // variants: 5 rows x 2 CTAs/SM (128 registers), 9 rows x 1 CTA/SM (168), 13 rows x 1 (128)
    template <class F> void with_tj(int, F&& f) const {
        if (tj == 13) f(std::integral_constant<int, 13>{}, std::integral_constant<int, 1>{});
        else if (tj == 9) f(std::integral_constant<int, 9>{}, std::integral_constant<int, 1>{});
        else f(std::integral_constant<int, 5>{}, std::integral_constant<int, 2>{});
    }

    int prepare(const zda_zone_desc& d, int pitch, char* fbase, size_t fstride, int opt_tj, int opt_chunk, int opt_cluster) {
        tj = choose_tj(d.Nphi, opt_tj);
        minb = tj > 5 ? 1 : 2;
        const size_t es = d.complex_fields ? 2 * sizeof(R) : sizeof(R);
        const int W = (int)(es / 4), VEC = (int)(16 / es), LO = (2 + VEC - 1) / VEC, TI_OUT = (31 - LO) * VEC;
        cuuint64_t dims[4] = {(cuuint64_t)d.Nr * W, (cuuint64_t)d.Nphi + 2 * field_ghost(d), (cuuint64_t)d.Nz, 12};
        cuuint64_t strides[3] = {(cuuint64_t)pitch * es, (cuuint64_t)pitch * (d.Nphi + 2 * field_ghost(d)) * es, (cuuint64_t)fstride};
        cuuint32_t box[4] = {FUSED_ROW_BYTES / 4, (cuuint32_t)tj + 4, 1, 3};
        cuuint32_t estr[4] = {1, 1, 1, 1};
        using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                      const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                      CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        ZDA_CUDA_OK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (fn == nullptr || qres != cudaDriverEntryPointSuccess)
            return fail(ZDA_E_CUDA, "cuTensorMapEncodeTiled is not available in this driver");
        CUresult r = reinterpret_cast<EncodeFn>(fn)(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, fbase, dims, strides, box, estr,
                                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(ZDA_E_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
        G.n_ti = (d.Nr + TI_OUT - 1) / TI_OUT;
        G.n_tj = (d.Nphi + tj - 1) / tj;
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        G.cluster = 1;
        if (opt_cluster >= 1 && opt_cluster <= 8) G.cluster = opt_cluster;
        if (G.n_tj == 1) G.cluster = 1;
        G.n_tjc = (G.n_tj + G.cluster - 1) / G.cluster;
        // z-chunks: each chunk recomputes three planes of step A below it, so chunks are longer than the one-step kernel's
        const long tiles = (long)G.n_ti * G.n_tjc * G.cluster, slots = (long)minb * sms;
        int nzc = std::max(1, (d.Nz + 31) / 63);
        if (tiles * nzc < 2 * slots) nzc = (int)std::min<long>((2 * slots + tiles - 1) / tiles, std::max(1, d.Nz / 12));
        int best_chunk = (d.Nz + nzc - 1) / nzc;
        if (opt_chunk > 0) best_chunk = std::min(opt_chunk, d.Nz);
        G.chunk = best_chunk;
        G.n_zc = (d.Nz + G.chunk - 1) / G.chunk;
        G.aE = 0; G.aH = 3;
        with_tj(tj, [&](auto c, auto) { smem_bytes = sizeof(Fused2Smem<decltype(c)::value>) + 1024; });
        char buf[200];
        snprintf(buf, sizeof(buf), "fused2(2 steps/pass, tma tile %dx%d of %dx%d, z-chunk %d, grid %ld x %d thr x %d/SM, cluster %d, smem %zu B)",
                 TI_OUT, tj, 32 * VEC, tj + 4, G.chunk, (long)G.n_ti * G.n_tjc * G.cluster * G.n_zc, (tj + 3) * 32, minb, G.cluster, smem_bytes);
        nm = buf;
        return ZDA_OK;
    }
    const char* name() const { return nm.c_str(); }

    template <class T> int launch(const StepParams<T>& P, int cur, cudaStream_t st) {
        int rc = ZDA_OK;
        with_tj(tj, [&](auto c, auto mb) { rc = launch_tj<T, decltype(c)::value, decltype(mb)::value>(P, cur, st); });
        return rc;
    }
    template <class T, int TJ, int MINB> int launch_tj(const StepParams<T>& P, int cur, cudaStream_t st) {
        constexpr int ci = ElemTraits<T>::cplx ? 1 : 0;
        auto kern = fused2_step_kernel<T, TJ, MINB>;
        if (!attr_done[ci]) {
            ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
            ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
            attr_done[ci] = true;
        }
        FusedGeom g = G;
        g.aE = cur * 6; g.aH = cur * 6 + 3;
        const unsigned grid = (unsigned)((long)G.n_ti * G.n_tjc * G.cluster * G.n_zc);
        if (G.cluster == 1) {
            kern<<<grid, (TJ + 3) * 32, smem_bytes, st>>>(P, tmap, g);
            return ZDA_OK;
        }
        cudaLaunchConfig_t cfg;
        std::memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3((TJ + 3) * 32);
        cfg.dynamicSmemBytes = smem_bytes; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)G.cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        ZDA_CUDA_OK(cudaLaunchKernelEx(&cfg, kern, P, tmap, g));
        return ZDA_OK;
    }
};

}  // namespace zda
