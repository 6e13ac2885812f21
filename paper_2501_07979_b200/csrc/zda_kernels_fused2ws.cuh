// Two time steps per HBM pass, warp-specialised (DESIGN.md 7.1b "what would make it pay").
//
// Same schedule, halo recompute and arithmetic as fused2_step_kernel, but the two steps live in DIFFERENT warps:
//
//   A-warps (one per tile row 0 .. TJ+2)   phase 1  H_A(k)    from the TMA rings          | interval 1
//                                          phase 2  E_A(k)                                 | interval 2
//   B-warps (one per tile row 1 .. TJ+1)   phase 3  H_B(k-2)  from the hand-over rings    | interval 1
//                                          phase 4  E_B(k-2), stores, running DFT         | interval 2
//
// A hands E_A(k) and H_A(k) (all three components) to B through shared-memory rings of three planes; B trails A by two
// planes, so both kinds of warp work between the same two __syncthreads of an iteration and nobody carries the other
// step's state: each warp needs the registers of a ONE-step kernel (128), and the CTA holds 2 TJ + 4 warps (16 at TJ = 6)
// instead of fused2's TJ + 3 at 168 registers.  The CPML auxiliaries after step A travel from A to B through a per-CTA
// scratch in global memory (slab planes and edge tiles only; L2-resident).
#pragma once
#include "zda_kernels_fused2.cuh"

namespace zda {

template <int TJ> struct alignas(1024) Fused2WsSmem {
    static constexpr int ROWS = TJ + 4;
    struct alignas(128) Slot { unsigned char c[3][ROWS][FUSED_ROW_BYTES]; };
    Slot E[3];                                                     // E^n planes k, k+1, k+2
    Slot H[2];                                                     // H^{n-1/2} planes k, k+1
    alignas(16) unsigned char HnA[2][TJ + 3][FUSED_PAY_BYTES];     // step A: new {Hr, Hz} of rows 0..TJ+2 (phase 2's y-1 neighbour)
    alignas(16) unsigned char EA[3][3][TJ + 3][FUSED_PAY_BYTES];   // hand-over: E_A planes kA, kA-1, kA-2, rows 1..TJ+2
    alignas(16) unsigned char HA[3][3][TJ + 2][FUSED_PAY_BYTES];   // hand-over: H_A planes, rows 1..TJ+1
    alignas(16) unsigned char HnB[2][TJ + 2][FUSED_PAY_BYTES];     // step B: new {Hr, Hz} of rows 1..TJ+1 (phase 4's y-1 neighbour)
    alignas(16) unsigned char coef[12][FUSED_PAY_BYTES];
    unsigned long long barE[3], barH[2];
};

// per-CTA scratch for the CPML auxiliaries after step A: [slot 3][array 8][row TJ+2][32 lanes x 16 B]
template <int TJ> constexpr size_t fused2ws_scratch_bytes() { return (size_t)3 * 8 * (TJ + 2) * FUSED_PAY_BYTES; }

template <class T, int TJ, bool RS>
__device__ __forceinline__ void fused2ws_body(const StepParams<T>& P, const CUtensorMap& tmap, const FusedGeom& G,
                                              unsigned char* __restrict__ scratch_all) {
    using R = typename ElemTraits<T>::Real;
    using V = VecT<T>;
    using Smem = Fused2WsSmem<TJ>;
    constexpr int VEC = V::N;
    constexpr int W = (int)sizeof(T) / 4;
    constexpr int NA = TJ + 3, NB = TJ + 1, NW = NA + NB;
    constexpr int LO = (2 + VEC - 1) / VEC;
    constexpr int NU_OUT = 31 - LO;
    constexpr int TI_OUT = NU_OUT * VEC;
    constexpr unsigned SLOT_BYTES = 3u * (TJ + 4) * FUSED_ROW_BYTES;

    extern __shared__ unsigned char smem_raw[];
    Smem& S = *reinterpret_cast<Smem*>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u));

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const bool roleA = warp < NA;
    int b = blockIdx.x;
    const int crank = b % G.cluster; b /= G.cluster;
    const int ti = b % G.n_ti; b /= G.n_ti;
    const int tj = (b % G.n_tjc) * G.cluster + crank;
    const int zc = b / G.n_tjc;
    const bool tile_ok = tj < G.n_tj;
    const int a0 = ti * TI_OUT - LO * VEC;
    const int j0 = tj * TJ;
    const int Nr = P.Nr, Nphi = P.Nphi, Nz = P.Nz, pitch = P.pitch;
    const int ka = zc * G.chunk, kb = min(ka + G.chunk, Nz);
    const int kEA0 = ka > 0 ? ka - 1 : 0;               // first plane of E_A / H_B
    const int kstart = ka > 1 ? ka - 2 : 0;             // first plane of H_A
    const int nit = kb - kstart + 2;                    // iteration it: step A on plane kstart + it, step B TWO below
    const int nE = min(kb + 1, Nz) - kstart + 1;
    const int nH = min(kb, Nz - 1) - kstart + 1;
    const size_t row = (size_t)pitch, plane = row * Nphi, fplane = P.fplane;
    const int npr = P.npr_lo + P.npr_hi;
    // one CTA per SM (512 threads, 183 KB of shared memory), so the SM id names a scratch slot nobody else uses
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    unsigned char* scratch = scratch_all + (size_t)smid * fused2ws_scratch_bytes<TJ>();

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
    const int y = roleA ? warp : warp - NA + 1;          // tile row; physical row j0 - 2 + y
    const int jraw = j0 - 2 + y;
    int jm = jraw % Nphi; if (jm < 0) jm += Nphi;
    const int j = jm;
    const bool rowHA = roleA && tile_ok && (jraw <= Nphi);                    // H_A: rows -2 .. Nphi
    const bool rowEA = rowHA && (y >= 1);                                     // E_A: rows -1 .. Nphi
    const bool rowHB = !roleA && tile_ok && (jraw <= Nphi - 1);               // H_B: rows -1 .. Nphi - 1 (y = 1 .. TJ+1)
    const bool own = rowHB && (y >= 2);                                       // E_B and the stores
    const bool j_last = (j == Nphi - 1), j_first = (j == 0);
    const int ig = a0 + lane * VEC;
    const bool col_ok = (ig >= 0) && (ig < pitch);
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
    const size_t pj = (size_t)j * row + (size_t)(col_ok ? ig : 0);
    int gro[2 * FIELD_GHOST_MAX];
    const int n_gh = ghost_row_offsets(j, Nphi, FIELD_GHOST_MAX, gro);
    const int g_off0 = n_gh > 0 ? gro[0] * pitch : 0;
    const size_t orr_step = (size_t)Nphi * npr;
    // scratch slot of this thread: arrays 0..3 = H-side psi (z0, z1, r0, r1), 4..7 = E-side; row y - 1, lane
    auto scr = [&](int slot, int arr) __attribute__((always_inline)) {
        return reinterpret_cast<V*>(scratch + ((size_t)(slot * 8 + arr) * (TJ + 2) + (y - 1)) * FUSED_PAY_BYTES) + lane;
    };
    // CTA-wide barrier reached from the two role loops (different program points: a named barrier with an explicit count)
    auto cta_bar = [&]() __attribute__((always_inline)) { asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory"); };

    const int it_a = min(max(max(P.npz_lo, 1) + 2 - kstart, 0), nit);      // kB = kstart + it - 2 < max(npz_lo, 1)
    const int it_b = min(max(Nz - P.npz_hi - kstart, it_a), nit);          // kA = kstart + it < Nz - npz_hi

    if (roleA) {
        // =====================================================================================================
        // step A: H_A(kA), E_A(kA); hands both to the B-warps through S.EA / S.HA (and the psi scratch)
        // =====================================================================================================
        T hr_km[VEC], hp_km[VEC];                            // H_A {r, phi} of the previous plane
#pragma unroll
        for (int e = 0; e < VEC; ++e) { hr_km[e] = zero_of<T>(); hp_km[e] = zero_of<T>(); }
        size_t orrA = ((size_t)kstart * Nphi + j) * npr;

        auto iterA = [&](auto zs_tag, const int it) __attribute__((always_inline)) {
            constexpr bool zs = decltype(zs_tag)::value;
            const int kA = kstart + it, slot = kA % 3;
            const bool doHA = kA < Nz && kA <= kb;
            const bool doEA = doHA && kA >= kEA0;
            const bool ghostA = (kA == Nz) && (kA <= kb);     // the virtual plane: E_A there is the PEC zero
            const int kzA = (zs && doHA) ? slab_index(kA, Nz, P.npz_lo, P.npz_hi) : -1;
            const bool kmA = doHA && (kA >= P.mk0 && kA < P.mk1);
            const size_t ozA = (size_t)(kzA >= 0 ? kzA : 0) * plane + pj;
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
            const R cbgA = doHA ? ldg_early(P.zc + ZC_CE_BG * Nz + kA) : R(0);
            R bzH = R(0), czH = R(0), ikzH = R(1), bzE = R(0), czE = R(0), ikzE = R(1);
            if (zs && kzA >= 0) {
                bzH = ldg_early(P.zc + ZC_B_H * Nz + kA); czH = ldg_early(P.zc + ZC_C_H * Nz + kA); ikzH = ldg_early(P.zc + ZC_IK_H * Nz + kA);
                bzE = ldg_early(P.zc + ZC_B_I * Nz + kA); czE = ldg_early(P.zc + ZC_C_I * Nz + kA); ikzE = ldg_early(P.zc + ZC_IK_I * Nz + kA);
            }
            if (doHA) {
                if (it == 0) mbar_wait(&S.barE[0], 0);
                mbar_wait(&S.barE[(it + 1) % 3], ((it + 1) / 3) & 1);
                mbar_wait(&S.barH[it & 1], (it >> 1) & 1);
            }
            const typename Smem::Slot& Ek = S.E[it % 3];
            const typename Smem::Slot& Ek1 = S.E[(it + 1) % 3];
            const typename Smem::Slot& Hk = S.H[it & 1];

            // ---------------- phase 1: H_A(kA), rows 0 .. TJ+2 ----------------
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
                    in.bz = bzH; in.cz = czH; in.ikz = ikzH;
                    in.zs = zs && (kzA >= 0); in.rs = RS && ir[e] >= 0; in.skip_hr = false;
                    in.br = in.cr = R(0); in.ikr = R(1);
                    if (RS) { in.br = coefv(6).v[e]; in.cr = coefv(7).v[e]; in.ikr = coefv(8).v[e]; }
                    h_update_voxel(in, hA[0].v[e], hA[1].v[e], hA[2].v[e], pzH[0].v[e], pzH[1].v[e], prH[0][e], prH[1][e]);
                }
                *reinterpret_cast<V*>(&S.HnA[0][y][16 * lane]) = hA[0];
                *reinterpret_cast<V*>(&S.HnA[1][y][16 * lane]) = hA[2];
                if (y >= 1 && y <= TJ + 1) {                 // hand-over to the B-warp of this row
                    *reinterpret_cast<V*>(&S.HA[slot][0][y][16 * lane]) = hA[0];
                    *reinterpret_cast<V*>(&S.HA[slot][1][y][16 * lane]) = hA[1];
                    *reinterpret_cast<V*>(&S.HA[slot][2][y][16 * lane]) = hA[2];
                    if (zs && kzA >= 0) { *scr(slot, 0) = pzH[0]; *scr(slot, 1) = pzH[1]; }
                    if (RS && any_rs) {
                        V t0, t1;
#pragma unroll
                        for (int e = 0; e < VEC; ++e) { t0.v[e] = prH[0][e]; t1.v[e] = prH[1][e]; }
                        *scr(slot, 2) = t0; *scr(slot, 3) = t1;
                    }
                }
            }
            cta_bar();
            if (tid == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                if (it + 3 < nE) issueE(it + 3);
                if (it + 2 < nH) issueH(it + 2);
            }

            // ---------------- phase 2: E_A(kA), rows 1 .. TJ+2 ----------------
            if (rowEA && (doEA || ghostA)) {
                V eA[3];
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int e = 0; e < VEC; ++e) eA[c].v[e] = zero_of<T>();
                if (doEA) {
                    V hr_jm = *reinterpret_cast<const V*>(&S.HnA[0][y - 1][16 * lane]);
                    V hz_jm = *reinterpret_cast<const V*>(&S.HnA[1][y - 1][16 * lane]);
                    if (j_first) {
#pragma unroll
                        for (int e = 0; e < VEC; ++e) {
                            hr_jm.v[e] = phase_mul(P.pr, -P.pi, hr_jm.v[e]);
                            hz_jm.v[e] = phase_mul(P.pr, -P.pi, hz_jm.v[e]);
                        }
                    }
                    T hp_w = shfl_up1(hA[1].v[VEC - 1]), hz_w = shfl_up1(hA[2].v[VEC - 1]);
                    if (lane == 0) { hp_w = zero_of<T>(); hz_w = zero_of<T>(); }
                    T jr[VEC], jp[VEC];
#pragma unroll
                    for (int e = 0; e < VEC; ++e) { jr[e] = zero_of<T>(); jp[e] = zero_of<T>(); }
                    if (kA == P.src_k && P.n_terms > 0 && P.n < P.tab_len && col_ok) {
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
                        in.hr_km = hr_km[e]; in.hp_km = hp_km[e];
                        in.hp_im = (e > 0) ? hA[1].v[(e + VEC - 1) % VEC] : hp_w;
                        in.hz_im = (e > 0) ? hA[2].v[(e + VEC - 1) % VEC] : hz_w;
                        in.jr = jr[e]; in.jp = jp[e];
                        in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.cc = c_cc.v[e]; in.cd = c_cd.v[e];
                        in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.cE = (kmA && col_ok) ? cEv[e] : cbgA;
                        in.bz = bzE; in.cz = czE; in.ikz = ikzE;
                        in.zs = zs && (kzA >= 0); in.rs = RS && ir[e] >= 0;
                        in.k_pos = zs ? (kA > 0) : true;
                        in.i_pos = RS ? (ig + e > 0) : true;
                        in.br = in.cr = R(0); in.ikr = R(1);
                        if (RS) { in.br = coefv(9).v[e]; in.cr = coefv(10).v[e]; in.ikr = coefv(11).v[e]; }
                        e_update_voxel(in, eA[0].v[e], eA[1].v[e], eA[2].v[e], pzE[0].v[e], pzE[1].v[e], prE[0][e], prE[1][e]);
                        if (RS && !in_dom[e]) { eA[0].v[e] = zero_of<T>(); eA[1].v[e] = zero_of<T>(); eA[2].v[e] = zero_of<T>(); }
                    }
                    if (y >= 2 && y <= TJ + 1) {             // E-side psi after step A, for the B-warp of this (own) row
                        if (zs && kzA >= 0) { *scr(slot, 4) = pzE[0]; *scr(slot, 5) = pzE[1]; }
                        if (RS && any_rs) {
                            V t0, t1;
#pragma unroll
                            for (int e = 0; e < VEC; ++e) { t0.v[e] = prE[0][e]; t1.v[e] = prE[1][e]; }
                            *scr(slot, 6) = t0; *scr(slot, 7) = t1;
                        }
                    }
                }
                *reinterpret_cast<V*>(&S.EA[slot][0][y][16 * lane]) = eA[0];
                *reinterpret_cast<V*>(&S.EA[slot][1][y][16 * lane]) = eA[1];
                *reinterpret_cast<V*>(&S.EA[slot][2][y][16 * lane]) = eA[2];
            }
            if (rowHA && doHA) {
#pragma unroll
                for (int e = 0; e < VEC; ++e) { hr_km[e] = hA[0].v[e]; hp_km[e] = hA[1].v[e]; }
            }
            orrA += orr_step;
            cta_bar();
        };
        int it = 0;
#pragma unroll 1
        for (; it < it_a; ++it) iterA(std::true_type{}, it);
#pragma unroll 1
        for (; it < it_b; ++it) iterA(std::false_type{}, it);
#pragma unroll 1
        for (; it < nit; ++it) iterA(std::true_type{}, it);
    } else {
        // =====================================================================================================
        // step B, two planes behind: H_B(kB), E_B(kB) from the hand-over rings; stores, ring copies, running DFT
        // =====================================================================================================
        T hBr_km[VEC], hBp_km[VEC];                          // H_B {r, phi} of the previous plane
#pragma unroll
        for (int e = 0; e < VEC; ++e) { hBr_km[e] = zero_of<T>(); hBp_km[e] = zero_of<T>(); }
        size_t foB = (size_t)(kstart - 2) * fplane + (size_t)(j + FIELD_GHOST_MAX) * row + (size_t)(col_ok ? ig : 0);
        size_t orrB = ((size_t)(kstart - 2) * Nphi + j) * npr;

        auto iterB = [&](auto zs_tag, const int it) __attribute__((always_inline)) {
            constexpr bool zs = decltype(zs_tag)::value;
            const int kB = kstart + it - 2;
            const int slot = (kB + 3) % 3, slot1 = (kB + 4) % 3;      // planes kB, kB + 1 (kB >= -2)
            const bool doHB = kB >= kEA0 && kB <= kb - 1;
            const bool doEB = kB >= ka && kB <= kb - 1;
            const int kzB = (zs && kB >= 0) ? slab_index(kB, Nz, P.npz_lo, P.npz_hi) : -1;
            const bool kmB = (kB >= P.mk0 && kB < P.mk1);
            const bool kdB = (kB >= P.dk0 && kB < P.dk1);
            const size_t ozB = (size_t)(kzB >= 0 ? kzB : 0) * plane + pj;
            const bool monB = (kB == P.mon_k) && (P.dft_mon != nullptr);
            const bool dboxB = kdB && (ig < P.di1) && (ig + VEC > P.di0);
            const bool dgrpB = dboxB && (P.dft_design != nullptr);
            R cEv[VEC];
#pragma unroll
            for (int e = 0; e < VEC; ++e) cEv[e] = R(0);
            if (own && doEB && col_ok) {
                if (kmB) {
                    struct alignas(VEC * sizeof(R)) CEV { R v[VEC]; };
                    const CEV c = ldg_early(reinterpret_cast<const CEV*>(P.cE_design + (size_t)(kB - P.mk0) * plane + pj));
#pragma unroll
                    for (int e = 0; e < VEC; ++e) cEv[e] = c.v[e];
                }
                if (out_lane && dgrpB) {
                    const int Ld = P.dk1 - P.dk0;
                    for (int fc = 0; fc < 3 * P.F; ++fc)
                        prefetch_l2(P.dft_design + ((size_t)fc * Ld + (kB - P.dk0)) * plane + pj);
                }
                if (out_lane && monB)
                    for (int fc = 0; fc < 3 * P.F; ++fc) prefetch_l2(P.dft_mon + (size_t)fc * plane + pj);
            }
            const R cbgB = (kB >= 0 && kB < Nz) ? ldg_early(P.zc + ZC_CE_BG * Nz + kB) : R(0);
            R bzH = R(0), czH = R(0), ikzH = R(1), bzE = R(0), czE = R(0), ikzE = R(1);
            if (zs && kzB >= 0) {
                bzH = ldg_early(P.zc + ZC_B_H * Nz + kB); czH = ldg_early(P.zc + ZC_C_H * Nz + kB); ikzH = ldg_early(P.zc + ZC_IK_H * Nz + kB);
                bzE = ldg_early(P.zc + ZC_B_I * Nz + kB); czE = ldg_early(P.zc + ZC_C_I * Nz + kB); ikzE = ldg_early(P.zc + ZC_IK_I * Nz + kB);
            }

            // ---------------- phase 3: H_B(kB), rows 1 .. TJ+1 ----------------
            V hB[3], eAp[3];
            V pzHB[2], pzEB[2];
            T prHB[2][VEC], prEB[2][VEC];
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int e = 0; e < VEC; ++e) { hB[c].v[e] = zero_of<T>(); eAp[c].v[e] = zero_of<T>(); }
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
                for (int e = 0; e < VEC; ++e) { pzHB[c].v[e] = pzEB[c].v[e] = zero_of<T>(); prHB[c][e] = prEB[c][e] = zero_of<T>(); }
            if (rowHB && doHB) {
                eAp[0] = *reinterpret_cast<const V*>(&S.EA[slot][0][y][16 * lane]);
                eAp[1] = *reinterpret_cast<const V*>(&S.EA[slot][1][y][16 * lane]);
                eAp[2] = *reinterpret_cast<const V*>(&S.EA[slot][2][y][16 * lane]);
                V er_jp = *reinterpret_cast<const V*>(&S.EA[slot][0][y + 1][16 * lane]);
                V ez_jp = *reinterpret_cast<const V*>(&S.EA[slot][2][y + 1][16 * lane]);
                if (j_last) {
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        er_jp.v[e] = phase_mul(P.pr, P.pi, er_jp.v[e]);
                        ez_jp.v[e] = phase_mul(P.pr, P.pi, ez_jp.v[e]);
                    }
                }
                const V er_kp = *reinterpret_cast<const V*>(&S.EA[slot1][0][y][16 * lane]);
                const V ep_kp = *reinterpret_cast<const V*>(&S.EA[slot1][1][y][16 * lane]);
                hB[0] = *reinterpret_cast<const V*>(&S.HA[slot][0][y][16 * lane]);
                hB[1] = *reinterpret_cast<const V*>(&S.HA[slot][1][y][16 * lane]);
                hB[2] = *reinterpret_cast<const V*>(&S.HA[slot][2][y][16 * lane]);
                if (zs && kzB >= 0) { pzHB[0] = *scr(slot, 0); pzHB[1] = *scr(slot, 1); }
                if (RS && any_rs) {
                    const V t0 = *scr(slot, 2), t1 = *scr(slot, 3);
#pragma unroll
                    for (int e = 0; e < VEC; ++e) { prHB[0][e] = t0.v[e]; prHB[1][e] = t1.v[e]; }
                }
                T ep_nx = shfl_down1(eAp[1].v[0]), ez_nx = shfl_down1(eAp[2].v[0]);
                if (lane == 31) { ep_nx = zero_of<T>(); ez_nx = zero_of<T>(); }
                const CoefV c_rI = coefv(0), c_rH = coefv(1), c_ca = coefv(2), c_cb = coefv(3);
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    HIn<T, R> in;
                    in.er = eAp[0].v[e]; in.ep = eAp[1].v[e]; in.ez = eAp[2].v[e];
                    in.er_jp = er_jp.v[e]; in.ez_jp = ez_jp.v[e];
                    in.er_kp = er_kp.v[e]; in.ep_kp = ep_kp.v[e];
                    in.ep_ip = (e + 1 < VEC) ? eAp[1].v[(e + 1) % VEC] : ep_nx;
                    in.ez_ip = (e + 1 < VEC) ? eAp[2].v[(e + 1) % VEC] : ez_nx;
                    in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.ca = c_ca.v[e]; in.cb = c_cb.v[e];
                    in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.dt = P.dt;
                    in.bz = bzH; in.cz = czH; in.ikz = ikzH;
                    in.zs = zs && (kzB >= 0); in.rs = RS && ir[e] >= 0; in.skip_hr = false;
                    in.br = in.cr = R(0); in.ikr = R(1);
                    if (RS) { in.br = coefv(6).v[e]; in.cr = coefv(7).v[e]; in.ikr = coefv(8).v[e]; }
                    h_update_voxel(in, hB[0].v[e], hB[1].v[e], hB[2].v[e], pzHB[0].v[e], pzHB[1].v[e], prHB[0][e], prHB[1][e]);
                }
                *reinterpret_cast<V*>(&S.HnB[0][y][16 * lane]) = hB[0];
                *reinterpret_cast<V*>(&S.HnB[1][y][16 * lane]) = hB[2];
            }
            cta_bar();

            // ---------------- phase 4: E_B(kB), own rows; stores ----------------
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
                T hp_w = shfl_up1(hB[1].v[VEC - 1]), hz_w = shfl_up1(hB[2].v[VEC - 1]);
                if (lane == 0) { hp_w = zero_of<T>(); hz_w = zero_of<T>(); }
                T jr[VEC], jp[VEC];
#pragma unroll
                for (int e = 0; e < VEC; ++e) { jr[e] = zero_of<T>(); jp[e] = zero_of<T>(); }
                if (kB == P.src_k && P.n_terms > 0 && P.n + 1 < P.tab_len && col_ok) {
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
                if (zs && kzB >= 0) { pzEB[0] = *scr(slot, 4); pzEB[1] = *scr(slot, 5); }
                if (RS && any_rs) {
                    const V t0 = *scr(slot, 6), t1 = *scr(slot, 7);
#pragma unroll
                    for (int e = 0; e < VEC; ++e) { prEB[0][e] = t0.v[e]; prEB[1][e] = t1.v[e]; }
                }
                V eB[3];
                eB[0] = eAp[0]; eB[1] = eAp[1]; eB[2] = eAp[2];
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
                    in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.cE = (kmB && col_ok) ? cEv[e] : cbgB;
                    in.bz = bzE; in.cz = czE; in.ikz = ikzE;
                    in.zs = zs && (kzB >= 0); in.rs = RS && ir[e] >= 0;
                    in.k_pos = zs ? (kB > 0) : true;
                    in.i_pos = RS ? (ig + e > 0) : true;
                    in.br = in.cr = R(0); in.ikr = R(1);
                    if (RS) { in.br = coefv(9).v[e]; in.cr = coefv(10).v[e]; in.ikr = coefv(11).v[e]; }
                    e_update_voxel(in, eB[0].v[e], eB[1].v[e], eB[2].v[e], pzEB[0].v[e], pzEB[1].v[e], prEB[0][e], prEB[1][e]);
                }
                if (out_lane) {
                    stg_vec(P.Hout[0] + foB, hB[0]); stg_vec(P.Hout[1] + foB, hB[1]); stg_vec(P.Hout[2] + foB, hB[2]);
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
#pragma unroll
                        for (int e = 0; e < VEC; ++e)
                            if (ir[e] >= 0) {
                                P.psiH_r_out[0][orrB + ir[e]] = prHB[0][e]; P.psiH_r_out[1][orrB + ir[e]] = prHB[1][e];
                                P.psiE_r_out[0][orrB + ir[e]] = prEB[0][e]; P.psiE_r_out[1][orrB + ir[e]] = prEB[1][e];
                            }
                    }
                    if (dboxB && P.ring_store != nullptr) {
                        const size_t Lp = (size_t)(P.dk1 - P.dk0) * plane;
                        T* rp = P.ring_store + (size_t)(kB - P.dk0) * plane + pj;
                        stg_vec(rp, eAp[0]); stg_vec(rp + Lp, eAp[1]); stg_vec(rp + 2 * Lp, eAp[2]);
                    }
                    if (dboxB && P.ring_store_b != nullptr) {
                        const size_t Lp = (size_t)(P.dk1 - P.dk0) * plane;
                        T* rp = P.ring_store_b + (size_t)(kB - P.dk0) * plane + pj;
                        stg_vec(rp, eB[0]); stg_vec(rp + Lp, eB[1]); stg_vec(rp + 2 * Lp, eB[2]);
                    }
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
            foB += fplane;
            orrB += orr_step;
            cta_bar();
        };
        int it = 0;
#pragma unroll 1
        for (; it < it_a; ++it) iterB(std::true_type{}, it);
#pragma unroll 1
        for (; it < it_b; ++it) iterB(std::false_type{}, it);
#pragma unroll 1
        for (; it < nit; ++it) iterB(std::true_type{}, it);
    }
}

template <class T, int TJ>
__global__ void __launch_bounds__((2 * TJ + 4) * 32, 1)
fused2ws_step_kernel(const __grid_constant__ StepParams<T> P, const __grid_constant__ CUtensorMap tmap, const FusedGeom G,
                     unsigned char* __restrict__ scratch) {
    constexpr int VEC = VecT<T>::N;
    constexpr int LO = (2 + VEC - 1) / VEC;
    constexpr int TI_OUT = (31 - LO) * VEC;
    const int a0 = (((int)blockIdx.x / G.cluster) % G.n_ti) * TI_OUT - LO * VEC;
    const bool tile_rs = (a0 < P.npr_lo) || (a0 + 32 * VEC > P.Nr - P.npr_hi) || (a0 <= 0) || (a0 + 32 * VEC > P.Nr);
    if (tile_rs) fused2ws_body<T, TJ, true>(P, tmap, G, scratch);
    else fused2ws_body<T, TJ, false>(P, tmap, G, scratch);
}

constexpr int FUSED2WS_TJ = 6;
constexpr int FUSED2WS_MAX_SMS = 256;        // scratch slots carved in the workspace (one per SM)
inline size_t fused2ws_workspace_bytes() { return (size_t)FUSED2WS_MAX_SMS * fused2ws_scratch_bytes<FUSED2WS_TJ>(); }

template <class R> size_t Fused2Plan<R>::ws_smem_bytes() { return sizeof(Fused2WsSmem<FUSED2WS_TJ>) + 1024; }
template <class R> template <class T> int Fused2Plan<R>::launch_ws(const StepParams<T>& P, int cur, cudaStream_t st) {
    constexpr int ci = ElemTraits<T>::cplx ? 1 : 0;
    static bool done[2] = {false, false};
    auto kern = fused2ws_step_kernel<T, FUSED2WS_TJ>;
    if (!done[ci]) {
        ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
        ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        done[ci] = true;
    }
    if (!ws_scratch) return fail(ZDA_E_STATE, "the warp-specialised kernel has no scratch");
    FusedGeom g = G;
    g.aE = cur * 6; g.aH = cur * 6 + 3;
    const unsigned grid = (unsigned)((long)G.n_ti * G.n_tjc * G.cluster * G.n_zc);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3((2 * FUSED2WS_TJ + 4) * 32);
    cfg.dynamicSmemBytes = smem_bytes; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)G.cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    ZDA_CUDA_OK(cudaLaunchKernelEx(&cfg, kern, P, tmap, g, ws_scratch));
    return ZDA_OK;
}

}  // namespace zda
