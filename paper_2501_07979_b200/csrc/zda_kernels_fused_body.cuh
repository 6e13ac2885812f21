// Body of the fused time-loop kernel and its host-side plan (see zda_kernels_fused.cuh for the design).
#pragma once
#include <type_traits>

namespace zda {

// RS: the tile (with its halo column) touches an r-CPML slab -- CTA-uniform, so interior tiles carry none of
// the r-slab code.  The per-plane body is instantiated for z-slab and non-slab planes the same way (ZS).
// XR: the zone carries the exact outer r-PML (R25) and this is an edge tile -- its own instantiation, so that every other
// tile (and every zone without it) runs exactly the code it ran before.
template <class T, int TJ, bool RS, bool XR = false>
__device__ __forceinline__ void fused_body(const StepParams<T>& P, const CUtensorMap& tmap, const FusedGeom& G, const int block_id) {
    using R = typename ElemTraits<T>::Real;
    using V = VecT<T>;
    using Smem = FusedSmem<TJ>;
    constexpr int VEC = V::N;
    constexpr int W = (int)sizeof(T) / 4;     // 32-bit words per element (the tensor map is in words)
    constexpr int TI = 32 * VEC;
    constexpr unsigned SLOT_BYTES = 3u * (TJ + 2) * FUSED_ROW_BYTES;

    extern __shared__ unsigned char smem_raw[];
    Smem& S = *reinterpret_cast<Smem*>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u));
    unsigned char (*coefx)[FUSED_PAY_BYTES] = reinterpret_cast<unsigned char (*)[FUSED_PAY_BYTES]>(reinterpret_cast<unsigned char*>(&S) + sizeof(Smem));

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // block index = (((zc * n_tjc + tjc) * n_ti + ti) * cluster + rank): a cluster is `cluster` phi-neighbouring tiles
    int b = block_id;       // blockIdx.x, or its index within the member of a batched launch
    const int crank = b % G.cluster; b /= G.cluster;
    const int ti = b % G.n_ti; b /= G.n_ti;
    const int tj = (b % G.n_tjc) * G.cluster + crank;
    const int zc = b / G.n_tjc;
    const bool tile_ok = tj < G.n_tj;          // padding CTAs of the last cluster only keep the cluster barrier company
    const int i0 = ti * TI, j0 = tj * TJ;
    const int Nr = P.Nr, Nphi = P.Nphi, Nz = P.Nz, pitch = P.pitch;
    const int ka = zc * G.chunk, kb = min(ka + G.chunk, Nz);
    const int kstart = ka > 0 ? ka - 1 : 0;   // a chunk that does not start at 0 first rebuilds H(ka - 1)
    const int nit = kb - kstart;
    const size_t row = (size_t)pitch, plane = row * Nphi, fplane = P.fplane;
    const int npr = P.npr_lo + P.npr_hi;

    auto issueE = [&](int e) __attribute__((always_inline)) {   // E planes kstart + e, e = 0..nit
        unsigned long long* bar = &S.barE[e % 3];
        mbar_expect_tx(bar, SLOT_BYTES);
        tma_load_4d(&S.E[e % 3], &tmap, bar, (i0 - VEC) * W, j0 + P.ghost - 1, kstart + e, G.aE);
    };
    auto issueH = [&](int h) __attribute__((always_inline)) {   // old H planes kstart + h, h = 0..nit-1
        unsigned long long* bar = &S.barH[h & 1];
        mbar_expect_tx(bar, SLOT_BYTES);
        tma_load_4d(&S.H[h & 1], &tmap, bar, (i0 - VEC) * W, j0 + P.ghost - 1, kstart + h, G.aH);
    };

    if (tid == 0) {
        for (int s = 0; s < 3; ++s) mbar_init(&S.barE[s], 1);
        for (int s = 0; s < 2; ++s) mbar_init(&S.barH[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int e = 0; e < 3 && e <= nit; ++e) issueE(e);
        for (int h = 0; h < 2 && h < nit; ++h) issueH(h);
    }
    // per-r curl coefficients of this tile -> shared memory (read back as vectors every plane: cheaper than
    // keeping 6 x VEC registers live across the whole z-march)
    {
        constexpr int tabs[18] = {RC_INV_RDPHI_INT, RC_INV_RDPHI_HALF, RC_CA, RC_CB, RC_CC, RC_CD,
                                  RC_B_H, RC_C_H, RC_IK_H, RC_B_I, RC_C_I, RC_IK_I,   // the r-CPML six only on edge tiles
                                  RC_BQ_I, RC_CQ_I, RC_BQ_H, RC_CQ_H, RC_HIR_I, RC_HIR_H};   // R25, edge tiles of an exact-PML zone
        for (int t = tid; t < (RS ? (XR ? 18 : 12) : 6) * TI; t += (TJ + 1) * 32) {
            const int w = t / TI, x = t % TI, idx = i0 + x;
            R* dst = w < 12 ? reinterpret_cast<R*>(S.coef[w]) : reinterpret_cast<R*>(coefx[w - 12]);
            dst[x] = idx < pitch ? P.rc[tabs[w] * pitch + idx] : R(0);
        }
    }
    __syncthreads();

    // ---- per-thread constants ---------------------------------------------------------------
    const int y = warp;                                  // tile row: 0 = halo row (physical j0 - 1), 1..TJ own
    const int jraw = j0 + y - 1;
    const int j = jraw < 0 ? Nphi - 1 : jraw;            // physical row (the first tile's halo row wraps)
    const bool row_ok = tile_ok && ((y == 0) || (jraw < Nphi));
    const bool own = (y > 0) && row_ok;
    const bool j_last = (j == Nphi - 1), j_first = (j == 0);
    const int ig = i0 + lane * VEC;                      // first column of this thread's 16 bytes
    const bool col_ok = ig < pitch;                      // pitch % 32 == 0: a group is all inside or all outside
    const bool in_nr = ig < Nr;

    struct alignas(VEC * sizeof(R)) CoefV { R v[VEC]; };
    auto coefv = [&](int w) __attribute__((always_inline)) {
        return w < 12 ? reinterpret_cast<const CoefV*>(S.coef[w])[lane] : reinterpret_cast<const CoefV*>(coefx[w - 12])[lane];
    };
    int ir[VEC];
    bool any_rs = false, xr[VEC], any_xr = false;      // xr: cell in the outer r-slab of an exact-PML zone (R25)
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
        const int idx = ig + e;
        ir[e] = (RS && idx < Nr) ? slab_index(idx, Nr, P.npr_lo, P.npr_hi) : -1;
        any_rs = any_rs || (ir[e] >= 0);
        xr[e] = XR && idx < Nr && idx >= Nr - P.npr_hi;
        any_xr = any_xr || xr[e];
    }

    T hr_km[VEC], hp_km[VEC];                            // H^{n+1/2}(k - 1) at this thread's sites
#pragma unroll
    for (int e = 0; e < VEC; ++e) { hr_km[e] = zero_of<T>(); hp_km[e] = zero_of<T>(); }

    // offsets that advance by a constant per plane (kept as running values instead of being rebuilt from k)
    const size_t pj = (size_t)j * row + ig;                            // (j, ig) in the dense [Nphi][pitch] arrays
    size_t fo = (size_t)kstart * fplane + (size_t)(j + P.ghost) * row + ig;  // (k, j, ig) in the ghost-row field layout
    size_t orr = ((size_t)kstart * Nphi + j) * npr;                    // (k, j, 0) in the r-slab psi arrays
    // ghost copies of this row (rows within FIELD_GHOST of the wrap; several when Nphi is tiny)
    int gro[2 * FIELD_GHOST_MAX];
    const int n_gh = ghost_row_offsets(j, Nphi, P.ghost, gro);
    // rows 0 / Nphi - 1 of a zone with Nphi >= 4 have exactly one copy each, rows 1 / Nphi - 2 one: keep the first offset
    // in a register and the rest (tiny Nphi only) behind a rare branch; in elements: at most (Nphi + 2) pitch < 2^31
    const int g_off0 = n_gh > 0 ? gro[0] * pitch : 0;
    const size_t orr_step = (size_t)Nphi * npr;

    auto plane_iter = [&](auto zs_tag, const int it) __attribute__((always_inline)) {
        constexpr bool zs = decltype(zs_tag)::value;
        const int k = kstart + it;
        const bool store = (k >= ka);
        const int kz = zs ? slab_index(k, Nz, P.npz_lo, P.npz_hi) : -1;
        const bool kd = (k >= P.dk0 && k < P.dk1);
        const bool km = (k >= P.mk0 && k < P.mk1);
        const size_t oz = (size_t)(zs ? kz : 0) * plane + pj;
        // Global operands of this plane that do not come through TMA are requested NOW, before waiting on
        // the tiles: z-slab psi (H and E side) and dt/eps of the design layer as loads, the DFT accumulators
        // as L2 prefetches.  Their DRAM latency then overlaps the TMA wait and the H phase.
        V pzH0, pzH1, pzE0, pzE1;
        R cEv[VEC];
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            pzH0.v[e] = pzH1.v[e] = pzE0.v[e] = pzE1.v[e] = zero_of<T>();
            cEv[e] = R(0);
        }
        if (zs && row_ok && col_ok) {
            pzH0 = ldg_early(reinterpret_cast<const V*>(P.psiH_z[0] + oz));
            pzH1 = ldg_early(reinterpret_cast<const V*>(P.psiH_z[1] + oz));
            if (own && store) {
                pzE0 = ldg_early(reinterpret_cast<const V*>(P.psiE_z[0] + oz));
                pzE1 = ldg_early(reinterpret_cast<const V*>(P.psiE_z[1] + oz));
            }
        }
        if (zs && row_ok && col_ok && k + 1 < kb) {   // next plane's z-slab psi -> L2, so that its loads above hit L2
            const int kz1 = slab_index(k + 1, Nz, P.npz_lo, P.npz_hi);
            if (kz1 >= 0) {
                const size_t o1 = (size_t)kz1 * plane + pj;
                prefetch_l2(P.psiH_z[0] + o1); prefetch_l2(P.psiH_z[1] + o1);
                if (own) { prefetch_l2(P.psiE_z[0] + o1); prefetch_l2(P.psiE_z[1] + o1); }
            }
        }
        // r-slab psi of this plane (edge tiles only)
        T prH0[VEC], prH1[VEC], prE0[VEC], prE1[VEC];
#pragma unroll
        for (int e = 0; e < VEC; ++e) prH0[e] = prH1[e] = prE0[e] = prE1[e] = zero_of<T>();
        T chH0[VEC], chH1[VEC], chE0[VEC], chE1[VEC];
#pragma unroll
        for (int e = 0; e < VEC; ++e) chH0[e] = chH1[e] = chE0[e] = chE1[e] = zero_of<T>();
        if (RS && any_rs && row_ok) {
#pragma unroll
            for (int e = 0; e < VEC; ++e)
                if (ir[e] >= 0) {
                    prH0[e] = ldg_early(P.psiH_r[0] + orr + ir[e]); prH1[e] = ldg_early(P.psiH_r[1] + orr + ir[e]);
                    if (XR && xr[e]) { chH0[e] = ldg_early(P.chiH[0] + orr + ir[e]); chH1[e] = ldg_early(P.chiH[1] + orr + ir[e]); }
                    if (own && store) {
                        prE0[e] = ldg_early(P.psiE_r[0] + orr + ir[e]); prE1[e] = ldg_early(P.psiE_r[1] + orr + ir[e]);
                        if (XR && xr[e]) { chE0[e] = ldg_early(P.chiE[0] + orr + ir[e]); chE1[e] = ldg_early(P.chiE[1] + orr + ir[e]); }
                    }
                }
        }
        const bool mon = (k == P.mon_k) && (P.dft_mon != nullptr) && (P.dft_mode != 0);
        const bool dbox = kd && (ig < P.di1) && (ig + VEC > P.di0);                        // group meets the design box
        const bool dgrp = dbox && (P.dft_mode != 0) && (P.dft_design != nullptr);
        const bool rgrp = dbox && (P.ring_store != nullptr);
        if (own && store && col_ok) {
            if (km) {
                struct alignas(VEC * sizeof(R)) CEV { R v[VEC]; };
                const CEV c = ldg_early(reinterpret_cast<const CEV*>(P.cE_design + (size_t)(k - P.mk0) * plane + pj));
#pragma unroll
                for (int e = 0; e < VEC; ++e) cEv[e] = c.v[e];
            }
            if (dgrp) {
                const int Ld = P.dk1 - P.dk0;
                for (int fc = 0; fc < 3 * P.F; ++fc)
                    prefetch_l2(P.dft_design + ((size_t)fc * Ld + (k - P.dk0)) * plane + pj);
            }
            if (mon && in_nr)
                for (int fc = 0; fc < 3 * P.F; ++fc) prefetch_l2(P.dft_mon + (size_t)fc * plane + pj);
        }
        // per-plane scalars: background dt/eps and, in a z-slab, the CPML coefficients at k + 1/2 and k
        const R cbg = ldg_early(P.zc + ZC_CE_BG * Nz + k);
        R bzH = R(0), czH = R(0), ikzH = R(1), bzE = R(0), czE = R(0), ikzE = R(1);
        if (zs) {
            bzH = ldg_early(P.zc + ZC_B_H * Nz + k); czH = ldg_early(P.zc + ZC_C_H * Nz + k); ikzH = ldg_early(P.zc + ZC_IK_H * Nz + k);
            bzE = ldg_early(P.zc + ZC_B_I * Nz + k); czE = ldg_early(P.zc + ZC_C_I * Nz + k); ikzE = ldg_early(P.zc + ZC_IK_I * Nz + k);
        }
        if (G.cluster > 1 && it > 0) cluster_wait();
        if (it == 0) mbar_wait(&S.barE[0], 0);
        mbar_wait(&S.barE[(it + 1) % 3], ((it + 1) / 3) & 1);
        mbar_wait(&S.barH[it & 1], (it >> 1) & 1);
        const typename Smem::Slot& Ek = S.E[it % 3];
        const typename Smem::Slot& Ek1 = S.E[(it + 1) % 3];
        const typename Smem::Slot& Hk = S.H[it & 1];
        const int buf = it & 1;

        // ================= H phase: rows 0..TJ =================
        V er, ep, ez, hrn, hpn, hzn;
        if (row_ok) {
            er = lds_vec<T>(Ek.c[0][y], lane + 1);
            ep = lds_vec<T>(Ek.c[1][y], lane + 1);
            ez = lds_vec<T>(Ek.c[2][y], lane + 1);
            const T ep_nx = lds_elem<T>(Ek.c[1][y], lane + 2, 0);
            const T ez_nx = lds_elem<T>(Ek.c[2][y], lane + 2, 0);
            V er_jp = lds_vec<T>(Ek.c[0][y + 1], lane + 1);
            V ez_jp = lds_vec<T>(Ek.c[2][y + 1], lane + 1);
            if (j_last) {
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    er_jp.v[e] = phase_mul(P.pr, P.pi, er_jp.v[e]);
                    ez_jp.v[e] = phase_mul(P.pr, P.pi, ez_jp.v[e]);
                }
            }
            const V er_kp = lds_vec<T>(Ek1.c[0][y], lane + 1);
            const V ep_kp = lds_vec<T>(Ek1.c[1][y], lane + 1);
            hrn = lds_vec<T>(Hk.c[0][y], lane + 1);
            hpn = lds_vec<T>(Hk.c[1][y], lane + 1);
            hzn = lds_vec<T>(Hk.c[2][y], lane + 1);

            V pz0 = pzH0, pz1 = pzH1;
            T pr0[VEC], pr1[VEC];
#pragma unroll
            for (int e = 0; e < VEC; ++e) { pr0[e] = prH0[e]; pr1[e] = prH1[e]; }
            const R bz = bzH, cz = czH, ikz = ikzH;
            const CoefV c_rI = coefv(0), c_rH = coefv(1), c_ca = coefv(2), c_cb = coefv(3);
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                HIn<T, R> in;
                in.er = er.v[e]; in.ep = ep.v[e]; in.ez = ez.v[e];
                in.er_jp = er_jp.v[e]; in.ez_jp = ez_jp.v[e];
                in.er_kp = er_kp.v[e]; in.ep_kp = ep_kp.v[e];
                in.ep_ip = (e + 1 < VEC) ? ep.v[(e + 1) % VEC] : ep_nx;
                in.ez_ip = (e + 1 < VEC) ? ez.v[(e + 1) % VEC] : ez_nx;
                in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.ca = c_ca.v[e]; in.cb = c_cb.v[e];
                in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.dt = P.dt;
                in.bz = bz; in.cz = cz; in.ikz = ikz;
                in.zs = zs; in.rs = RS && ir[e] >= 0; in.skip_hr = false;
                in.br = in.cr = R(0); in.ikr = R(1);
                if (RS) { in.br = coefv(6).v[e]; in.cr = coefv(7).v[e]; in.ikr = coefv(8).v[e]; }
                in.xr = XR && xr[e];
                if (XR && any_xr) {
                    in.bq_i = coefv(12).v[e]; in.cq_i = coefv(13).v[e]; in.bq_h = coefv(14).v[e]; in.cq_h = coefv(15).v[e];
                    in.hir = coefv(17).v[e];
                }
                if (XR) h_update_voxel(in, hrn.v[e], hpn.v[e], hzn.v[e], pz0.v[e], pz1.v[e], pr0[e], pr1[e], chH0[e], chH1[e]);
                else h_update_voxel(in, hrn.v[e], hpn.v[e], hzn.v[e], pz0.v[e], pz1.v[e], pr0[e], pr1[e]);
            }
            // new {Hr, Hz} of this row for the row above (E-update needs them at j - 1)
            *reinterpret_cast<V*>(&S.Hn[buf][0][y][16 * lane]) = hrn;
            *reinterpret_cast<V*>(&S.Hn[buf][1][y][16 * lane]) = hzn;
            if (own && store && in_nr) {
                stg_vec(P.Hout[0] + fo, hrn); stg_vec(P.Hout[1] + fo, hpn); stg_vec(P.Hout[2] + fo, hzn);
                if (n_gh > 0) {
                    stg_vec(P.Hout[0] + fo + (ptrdiff_t)g_off0, hrn); stg_vec(P.Hout[1] + fo + (ptrdiff_t)g_off0, hpn); stg_vec(P.Hout[2] + fo + (ptrdiff_t)g_off0, hzn);
                    for (int g = 1; g < n_gh; ++g) {
                        const ptrdiff_t o = (ptrdiff_t)gro[g] * (ptrdiff_t)row;
                        stg_vec(P.Hout[0] + fo + o, hrn); stg_vec(P.Hout[1] + fo + o, hpn); stg_vec(P.Hout[2] + fo + o, hzn);
                    }
                }
                if (zs) { stg_vec(P.psiH_z_out[0] + oz, pz0); stg_vec(P.psiH_z_out[1] + oz, pz1); }
                if (any_rs) {
#pragma unroll
                    for (int e = 0; e < VEC; ++e)
                        if (ir[e] >= 0) {
                            P.psiH_r_out[0][orr + ir[e]] = pr0[e]; P.psiH_r_out[1][orr + ir[e]] = pr1[e];
                            if (XR && xr[e]) { P.chiH_out[0][orr + ir[e]] = chH0[e]; P.chiH_out[1][orr + ir[e]] = chH1[e]; }
                        }
                }
            }
        }
        // halo column i0 - 1 (warp 0, one site per lane): new {Hphi, Hz} for the E-update at i0
        if (warp == 0 && i0 > 0 && lane < TJ && j0 + lane < Nphi) {
            const int yy = lane + 1, jj = j0 + lane, ic = i0 - 1;
            HIn<T, R> in;
            in.er = lds_elem<T>(Ek.c[0][yy], 0, VEC - 1);
            in.ep = lds_elem<T>(Ek.c[1][yy], 0, VEC - 1);
            in.ez = lds_elem<T>(Ek.c[2][yy], 0, VEC - 1);
            in.ep_ip = lds_elem<T>(Ek.c[1][yy], 1, 0);
            in.ez_ip = lds_elem<T>(Ek.c[2][yy], 1, 0);
            in.er_jp = lds_elem<T>(Ek.c[0][yy + 1], 0, VEC - 1);
            in.ez_jp = lds_elem<T>(Ek.c[2][yy + 1], 0, VEC - 1);
            if (jj == Nphi - 1) { in.er_jp = phase_mul(P.pr, P.pi, in.er_jp); in.ez_jp = phase_mul(P.pr, P.pi, in.ez_jp); }
            in.er_kp = lds_elem<T>(Ek1.c[0][yy], 0, VEC - 1);
            in.ep_kp = lds_elem<T>(Ek1.c[1][yy], 0, VEC - 1);
            T h0 = lds_elem<T>(Hk.c[0][yy], 0, VEC - 1);
            T h1 = lds_elem<T>(Hk.c[1][yy], 0, VEC - 1);
            T h2 = lds_elem<T>(Hk.c[2][yy], 0, VEC - 1);
            in.inv_rdphi_int = P.rc[RC_INV_RDPHI_INT * pitch + ic];
            in.inv_rdphi_half = P.rc[RC_INV_RDPHI_HALF * pitch + ic];
            in.ca = P.rc[RC_CA * pitch + ic]; in.cb = P.rc[RC_CB * pitch + ic];
            in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.dt = P.dt;
            in.skip_hr = false;
            in.zs = zs; in.bz = in.cz = R(0); in.ikz = R(1);
            T q0 = zero_of<T>(), q1 = zero_of<T>(), q2 = zero_of<T>(), q3 = zero_of<T>();
            if (zs) {
                in.bz = bzH; in.cz = czH; in.ikz = ikzH;
                const size_t o = (size_t)kz * plane + (size_t)jj * row + ic;
                q0 = P.psiH_z[0][o]; q1 = P.psiH_z[1][o];
            }
            const int irc = RS ? slab_index(ic, Nr, P.npr_lo, P.npr_hi) : -1;
            in.rs = irc >= 0; in.br = in.cr = R(0); in.ikr = R(1);
            T x0 = zero_of<T>(), x1 = zero_of<T>();
            if (in.rs) {
                in.br = P.rc[RC_B_H * pitch + ic]; in.cr = P.rc[RC_C_H * pitch + ic]; in.ikr = P.rc[RC_IK_H * pitch + ic];
                const size_t o = ((size_t)k * Nphi + jj) * npr + irc;
                q2 = P.psiH_r[0][o]; q3 = P.psiH_r[1][o];
                in.xr = XR && ic >= Nr - P.npr_hi;
                if (XR && in.xr) {
                    x0 = P.chiH[0][o]; x1 = P.chiH[1][o];
                    in.bq_i = P.rc[RC_BQ_I * pitch + ic]; in.cq_i = P.rc[RC_CQ_I * pitch + ic];
                    in.bq_h = P.rc[RC_BQ_H * pitch + ic]; in.cq_h = P.rc[RC_CQ_H * pitch + ic]; in.hir = P.rc[RC_HIR_H * pitch + ic];
                }
            }
            if (XR) h_update_voxel(in, h0, h1, h2, q0, q1, q2, q3, x0, x1);
            else h_update_voxel(in, h0, h1, h2, q0, q1, q2, q3);
            *reinterpret_cast<T*>(&S.Hcol[buf][0][lane][0]) = h1;
            *reinterpret_cast<T*>(&S.Hcol[buf][1][lane][0]) = h2;
        }
        // r-neighbours of the new H for the E phase: requested here so that the shuffle latency overlaps the barrier
        T hp_sh = zero_of<T>(), hz_sh = zero_of<T>();
        if (row_ok) { hp_sh = shfl_up1(hpn.v[VEC - 1]); hz_sh = shfl_up1(hzn.v[VEC - 1]); }
        __syncthreads();
        // E(k) and old H(k) have been consumed by every warp: refill their slots two planes ahead
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            if (it + 3 <= nit) issueE(it + 3);
            if (it + 2 < nit) issueH(it + 2);
        }

        // ================= E phase: own rows =================
        if (own) {
            if (store) {
                V hr_jm = *reinterpret_cast<const V*>(&S.Hn[buf][0][y - 1][16 * lane]);
                V hz_jm = *reinterpret_cast<const V*>(&S.Hn[buf][1][y - 1][16 * lane]);
                if (j_first) {
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        hr_jm.v[e] = phase_mul(P.pr, -P.pi, hr_jm.v[e]);
                        hz_jm.v[e] = phase_mul(P.pr, -P.pi, hz_jm.v[e]);
                    }
                }
                T hp_w = hp_sh, hz_w = hz_sh;
                if (lane == 0) {
                    hp_w = *reinterpret_cast<const T*>(&S.Hcol[buf][0][y - 1][0]);
                    hz_w = *reinterpret_cast<const T*>(&S.Hcol[buf][1][y - 1][0]);
                }
                R cE[VEC];
#pragma unroll
                for (int e = 0; e < VEC; ++e) cE[e] = (km && col_ok) ? cEv[e] : cbg;
                T jr[VEC], jp[VEC];
#pragma unroll
                for (int e = 0; e < VEC; ++e) { jr[e] = zero_of<T>(); jp[e] = zero_of<T>(); }
                if (k == P.src_k && P.n_terms > 0 && P.n < P.tab_len && col_ok) {
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
                V pz0 = pzE0, pz1 = pzE1;
                T pr0[VEC], pr1[VEC];
#pragma unroll
                for (int e = 0; e < VEC; ++e) { pr0[e] = prE0[e]; pr1[e] = prE1[e]; }
                const R bz = bzE, cz = czE, ikz = ikzE;
                const CoefV c_rI = coefv(0), c_rH = coefv(1), c_cc = coefv(4), c_cd = coefv(5);
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    EIn<T, R> in;
                    in.hr = hrn.v[e]; in.hp = hpn.v[e]; in.hz = hzn.v[e];
                    in.hr_jm = hr_jm.v[e]; in.hz_jm = hz_jm.v[e];
                    in.hr_km = hr_km[e]; in.hp_km = hp_km[e];
                    in.hp_im = (e > 0) ? hpn.v[(e + VEC - 1) % VEC] : hp_w;
                    in.hz_im = (e > 0) ? hzn.v[(e + VEC - 1) % VEC] : hz_w;
                    in.jr = jr[e]; in.jp = jp[e];
                    in.inv_rdphi_int = c_rI.v[e]; in.inv_rdphi_half = c_rH.v[e]; in.cc = c_cc.v[e]; in.cd = c_cd.v[e];
                    in.inv_dr = P.inv_dr; in.inv_dz = P.inv_dz; in.cE = cE[e];
                    in.bz = bz; in.cz = cz; in.ikz = ikz;
                    in.zs = zs; in.rs = RS && ir[e] >= 0;
                    in.k_pos = zs ? (k > 0) : true;       // plane 0 is always handled by the z-slab body (it_a below)
                    in.i_pos = (ig + e > 0);
                    in.br = in.cr = R(0); in.ikr = R(1);
                    if (RS) { in.br = coefv(9).v[e]; in.cr = coefv(10).v[e]; in.ikr = coefv(11).v[e]; }
                    in.xr = XR && xr[e];
                    if (XR && any_xr) {
                        in.bq_i = coefv(12).v[e]; in.cq_i = coefv(13).v[e]; in.bq_h = coefv(14).v[e]; in.cq_h = coefv(15).v[e];
                        in.hir = coefv(16).v[e];
                    }
                    if (XR) e_update_voxel(in, er.v[e], ep.v[e], ez.v[e], pz0.v[e], pz1.v[e], pr0[e], pr1[e], chE0[e], chE1[e]);
                    else e_update_voxel(in, er.v[e], ep.v[e], ez.v[e], pz0.v[e], pz1.v[e], pr0[e], pr1[e]);
                }
                if (in_nr) {
                    stg_vec(P.Eout[0] + fo, er); stg_vec(P.Eout[1] + fo, ep); stg_vec(P.Eout[2] + fo, ez);
                    if (n_gh > 0) {
                        stg_vec(P.Eout[0] + fo + (ptrdiff_t)g_off0, er); stg_vec(P.Eout[1] + fo + (ptrdiff_t)g_off0, ep); stg_vec(P.Eout[2] + fo + (ptrdiff_t)g_off0, ez);
                        for (int g = 1; g < n_gh; ++g) {
                            const ptrdiff_t o = (ptrdiff_t)gro[g] * (ptrdiff_t)row;
                            stg_vec(P.Eout[0] + fo + o, er); stg_vec(P.Eout[1] + fo + o, ep); stg_vec(P.Eout[2] + fo + o, ez);
                        }
                    }
                    if (zs) { stg_vec(P.psiE_z_out[0] + oz, pz0); stg_vec(P.psiE_z_out[1] + oz, pz1); }
                    if (any_rs) {
#pragma unroll
                        for (int e = 0; e < VEC; ++e)
                            if (ir[e] >= 0) {
                                P.psiE_r_out[0][orr + ir[e]] = pr0[e]; P.psiE_r_out[1][orr + ir[e]] = pr1[e];
                                if (XR && xr[e]) { P.chiE_out[0][orr + ir[e]] = chE0[e]; P.chiE_out[1][orr + ir[e]] = chE1[e]; }
                            }
                    }
                    if (rgrp) {     // keep this step's design-layer E for the accumulator visit s - 1 .. 2 launches from now
                        const size_t Lp = (size_t)(P.dk1 - P.dk0) * plane;
                        T* rp = P.ring_store + (size_t)(k - P.dk0) * plane + pj;
                        stg_vec(rp, er); stg_vec(rp + Lp, ep); stg_vec(rp + 2 * Lp, ez);
                    }
                    // running DFT (R8): Ehat_{c,f} += tw_f E_c^{n+1}; whole 16-byte groups (entries of a group
                    // that fall outside the design box / beyond Nr are scratch that nothing reads)
                    if (dgrp || mon) {
                        const int Ld = P.dk1 - P.dk0;
                        const bool two = (P.dft_mode == 2);
                        V o0, o1, o2;   // E^n of this site: the launch's input, intact in the other time buffer
#pragma unroll
                        for (int e = 0; e < VEC; ++e) o0.v[e] = o1.v[e] = o2.v[e] = zero_of<T>();
                        if (two) { o0 = ldg_vec(P.E[0] + fo); o1 = ldg_vec(P.E[1] + fo); o2 = ldg_vec(P.E[2] + fo); }
                        for (int f = 0; f < P.F; ++f) {
                            const Cx<R> tw = P.tw[(size_t)P.n * P.F + f];
                            const Cx<R> twp = two ? P.tw[(size_t)(P.n - 1) * P.F + f] : Cx<R>{R(0), R(0)};
                            if (dgrp)
                                dft_accumulate<T, R, VEC>(P.dft_design + ((size_t)f * 3 * Ld + (k - P.dk0)) * plane + pj,
                                                          (size_t)Ld * plane, twp, o0, o1, o2, tw, er, ep, ez);
                            if (mon)
                                dft_accumulate<T, R, VEC>(P.dft_mon + (size_t)f * 3 * plane + pj, plane, twp, o0, o1, o2,
                                                          tw, er, ep, ez);
                        }
                    }
                }
            }
#pragma unroll
            for (int e = 0; e < VEC; ++e) { hr_km[e] = hrn.v[e]; hp_km[e] = hpn.v[e]; }
        }
        fo += fplane;
        orr += orr_step;
        if (G.cluster > 1 && it + 1 < nit) cluster_arrive();
    };
    // three consecutive plane ranges: low z-slab, interior, high z-slab (each its own loop, so that the
    // slab / non-slab bodies do not meet at a per-plane branch)
    const int it_a = min(max(max(P.npz_lo, 1) - kstart, 0), nit);    // slab planes, and plane 0 (PEC predicate)
    const int it_b = min(max(Nz - P.npz_hi - kstart, it_a), nit);
    int it = 0;
#pragma unroll 1
    for (; it < it_a; ++it) plane_iter(std::true_type{}, it);
#pragma unroll 1
    for (; it < it_b; ++it) plane_iter(std::false_type{}, it);
#pragma unroll 1
    for (; it < nit; ++it) plane_iter(std::true_type{}, it);
}

template <class T, int TJ>
__global__ void __launch_bounds__((TJ + 1) * 32, 2)
fused_step_kernel(const __grid_constant__ StepParams<T> P, const __grid_constant__ CUtensorMap tmap, const FusedGeom G) {
    constexpr int TI = 32 * VecT<T>::N;
    const int i0 = (((int)blockIdx.x / G.cluster) % G.n_ti) * TI;
    const bool tile_rs = (i0 - 1 < P.npr_lo) || (i0 + TI > P.Nr - P.npr_hi);   // CTA-uniform
    if (tile_rs) fused_body<T, TJ, true>(P, tmap, G, (int)blockIdx.x);
    else fused_body<T, TJ, false>(P, tmap, G, (int)blockIdx.x);
}
// The same kernel for zones with the exact outer r-PML (R25): a kernel of its own, so that its extra edge-tile body does
// not sit in the instruction stream (and the instruction cache) of every other zone's launches.
template <class T, int TJ>
__global__ void __launch_bounds__((TJ + 1) * 32, 2)
fused_step_xr_kernel(const __grid_constant__ StepParams<T> P, const __grid_constant__ CUtensorMap tmap, const FusedGeom G) {
    constexpr int TI = 32 * VecT<T>::N;
    const int i0 = (((int)blockIdx.x / G.cluster) % G.n_ti) * TI;
    const bool tile_rs = (i0 - 1 < P.npr_lo) || (i0 + TI > P.Nr - P.npr_hi);
    if (tile_rs) fused_body<T, TJ, true, true>(P, tmap, G, (int)blockIdx.x);
    else fused_body<T, TJ, false>(P, tmap, G, (int)blockIdx.x);
}

// NEXT-4 ("a normally incident plane wave can be decomposed into m = +-1 components"): the members of a batch
// -- the m = +1 and m = -1 zones of a pair, or any zones of one shape and one launch plan -- advance one time step in
// ONE launch.  The member comes from the block index; each member brings its own parameter block (fields, psi, DFT
// accumulators, sheets, phase) and tensor map; geometry, plan and step index are common.  A thin wedge that fills half
// a wave of CTAs alone (config6: 280 CTAs on 296 slots) then fills the machine.
constexpr int FUSED_MAX_BATCH = 2;
template <class T> struct BatchParams {
    StepParams<T> m[FUSED_MAX_BATCH];
    CUtensorMap tmap[FUSED_MAX_BATCH];
};
template <class T, int TJ>
__global__ void __launch_bounds__((TJ + 1) * 32, 2)
fused_step_batch_kernel(const __grid_constant__ BatchParams<T> B, const FusedGeom G, const int ctas_per_member) {
    constexpr int TI = 32 * VecT<T>::N;
    const int member = (int)blockIdx.x / ctas_per_member, block_id = (int)blockIdx.x - member * ctas_per_member;
    const StepParams<T>& P = B.m[member];
    const int i0 = ((block_id / G.cluster) % G.n_ti) * TI;
    const bool tile_rs = (i0 - 1 < P.npr_lo) || (i0 + TI > P.Nr - P.npr_hi);
    if (tile_rs) fused_body<T, TJ, true>(P, B.tmap[member], G, block_id);
    else fused_body<T, TJ, false>(P, B.tmap[member], G, block_id);
}

// ---- host side -------------------------------------------------------------------------------------

template <class R> struct FusedPlan {
    CUtensorMap tmap;
    FusedGeom G;
    int tj = FUSED_TJ;      // tile rows per CTA, one of FUSED_TJ_MIN..FUSED_TJ_MAX (choose_tj)
    size_t smem_bytes = 0;
    std::string nm;
    bool attr_done[2] = {false, false};

    static bool supported(const zda_zone_desc& d) { return !d.has_axis; }

    // Thin wedges (Nphi ~ 7..16) pay for the phi tiling twice: the last tile is partly empty and every
    // tile carries one halo warp.  Warp-rows issued per plane = ceil(Nphi / TJ) (TJ + 1); take the TJ that minimises
    // it (ties: the larger tile).  Wide zones keep the measured-best 7.
    static int choose_tj(int Nphi, int opt_tj) {
        if (opt_tj == 6 || opt_tj == 7) return opt_tj;
        if (Nphi >= 64) return FUSED_TJ;
        int best = FUSED_TJ, best_cost = ((Nphi + FUSED_TJ - 1) / FUSED_TJ) * (FUSED_TJ + 1);
        for (int t = FUSED_TJ; t >= FUSED_TJ_MIN; --t) {
            const int cost = ((Nphi + t - 1) / t) * (t + 1);
            if (cost < best_cost) { best = t; best_cost = cost; }
        }
        return best;
    }
    template <class F> static void with_tj(int tj, F&& f) {
        switch (tj) {
            case 6: f(std::integral_constant<int, 6>{}); break;
            default: f(std::integral_constant<int, 7>{}); break;
        }
    }

    // opt_*: zda_set_option overrides (0 = the plan's own choice)
    int prepare(const zda_zone_desc& d, int pitch, char* fbase, size_t fstride, int opt_tj, int opt_chunk, int opt_cluster) {
        tj = choose_tj(d.Nphi, opt_tj);
        const size_t es = d.complex_fields ? 2 * sizeof(R) : sizeof(R);
        const int W = (int)(es / 4), VEC = (int)(16 / es), TI = 32 * VEC;
        cuuint64_t dims[4] = {(cuuint64_t)d.Nr * W, (cuuint64_t)d.Nphi + 2 * field_ghost(d), (cuuint64_t)d.Nz, 12};
        cuuint64_t strides[3] = {(cuuint64_t)pitch * es, (cuuint64_t)pitch * (d.Nphi + 2 * field_ghost(d)) * es, (cuuint64_t)fstride};
        cuuint32_t box[4] = {FUSED_ROW_BYTES / 4, (cuuint32_t)tj + 2, 1, 3};
        cuuint32_t estr[4] = {1, 1, 1, 1};
        // the driver entry point is looked up at run time so that libzda.so does not link against libcuda
        // (it must load, for the symbol check, on a machine without a driver)
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
        G.n_ti = (d.Nr + TI - 1) / TI;
        G.n_tj = (d.Nphi + tj - 1) / tj;
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        G.cluster = 2;   // measured on config2 / config4 (Gvox/s): 1 -> 81.1 / 69.1, 2 -> 82.8 / 71.7, 4 -> 79.2 / 72.2, 8 -> 72.5 / 69.1
        if (G.n_tj == 1) G.cluster = 1;
        if (opt_cluster >= 1 && opt_cluster <= 8) G.cluster = opt_cluster;
        G.n_tjc = (G.n_tj + G.cluster - 1) / G.cluster;
        // z-chunking.  Planes do not cost the same (z-CPML slabs, the design layer with its DFT accumulators), so long
        // chunks leave the heavy ones running alone at the end and bunch the accumulator traffic; chunks of about 28
        // planes let the CTA scheduler mix them, for one rebuilt plane in 28.  Measured (Gvox/s, chunk 20/25/32/42/63/125):
        // config4 76.2/76.3/76.3/76.4/75.1/71.8; config3 (16/20/25/29/34/100) 48.1/48.5/48.5/48.5/48.4/45.8; config2
        // (20/27/32/40/80/160) 86.0/86.3/85.9/85.5/82.5/72.7.  A zone too small for that still gets about two waves of
        // CTAs (config6, chunk 8/12/16/23: 29.2/29.9/26.7/27.3), chunks no shorter than 8 planes.
        const long tiles = (long)G.n_ti * G.n_tjc * G.cluster, slots = 2L * sms;   // CTAs per z-chunk
        int nzc = std::max(1, (d.Nz + 14) / 28);
        if (tiles * nzc < 2 * slots) nzc = (int)std::min<long>((2 * slots + tiles - 1) / tiles, std::max(1, d.Nz / 8));
        int best_chunk = (d.Nz + nzc - 1) / nzc;
        if (opt_chunk > 0) best_chunk = std::min(opt_chunk, d.Nz);
        G.chunk = best_chunk;
        G.n_zc = (d.Nz + G.chunk - 1) / G.chunk;
        G.aE = 0; G.aH = 3;
        with_tj(tj, [&](auto c) { smem_bytes = sizeof(FusedSmem<decltype(c)::value>) + 1024 + (d.rpml_exact ? 6 * FUSED_PAY_BYTES : 0); });
        char buf[160];
        snprintf(buf, sizeof(buf), "fused(tma tile %dx%d, z-chunk %d, grid %ld x %d thr, cluster %d, smem %zu B)", TI, tj,
                 G.chunk, (long)G.n_ti * G.n_tjc * G.cluster * G.n_zc, (tj + 1) * 32, G.cluster, smem_bytes);
        nm = buf;
        return ZDA_OK;
    }
    const char* name() const { return nm.c_str(); }

    template <class T> int launch(const StepParams<T>& P, int cur, cudaStream_t st) {
        int rc = ZDA_OK;
        with_tj(tj, [&](auto c) { rc = launch_tj<T, decltype(c)::value>(P, cur, st); });
        return rc;
    }
    // One launch for two zones of the same shape and plan (this plan's geometry; `other` supplies its tensor map).
    bool batch_attr_done[2] = {false, false};
    template <class T> int launch_batch(const StepParams<T>& P0, const StepParams<T>& P1, const FusedPlan& other, int cur, cudaStream_t st) {
        int rc = ZDA_OK;
        with_tj(tj, [&](auto c) { rc = launch_batch_tj<T, decltype(c)::value>(P0, P1, other, cur, st); });
        return rc;
    }
    template <class T, int TJ> int launch_batch_tj(const StepParams<T>& P0, const StepParams<T>& P1, const FusedPlan& other, int cur,
                                                   cudaStream_t st) {
        constexpr int ci = ElemTraits<T>::cplx ? 1 : 0;
        auto kern = fused_step_batch_kernel<T, TJ>;
        if (!batch_attr_done[ci]) {
            ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
            ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
            batch_attr_done[ci] = true;
        }
        BatchParams<T> B;
        B.m[0] = P0; B.m[1] = P1;
        B.tmap[0] = tmap; B.tmap[1] = other.tmap;
        FusedGeom g = G;
        g.aE = cur * 6; g.aH = cur * 6 + 3;
        const int per = (int)((long)G.n_ti * G.n_tjc * G.cluster * G.n_zc);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(2u * (unsigned)per); cfg.blockDim = dim3((TJ + 1) * 32);
        cfg.dynamicSmemBytes = smem_bytes; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)G.cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        ZDA_CUDA_OK(cudaLaunchKernelEx(&cfg, kern, B, g, per));
        return ZDA_OK;
    }
    template <class T, int TJ> int launch_tj(const StepParams<T>& P, int cur, cudaStream_t st) {
        constexpr int ci = ElemTraits<T>::cplx ? 1 : 0;
        auto kern = P.rpml_exact ? fused_step_xr_kernel<T, TJ> : fused_step_kernel<T, TJ>;
        if (!attr_done[ci]) {
            ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
            ZDA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
            attr_done[ci] = true;
        }
        FusedGeom g = G;
        g.aE = cur * 6; g.aH = cur * 6 + 3;
        const unsigned grid = (unsigned)((long)G.n_ti * G.n_tjc * G.cluster * G.n_zc);
        if (G.cluster == 1) {
            kern<<<grid, (TJ + 1) * 32, smem_bytes, st>>>(P, tmap, g);
            return ZDA_OK;
        }
        cudaLaunchConfig_t cfg;
        std::memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3((TJ + 1) * 32);
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
