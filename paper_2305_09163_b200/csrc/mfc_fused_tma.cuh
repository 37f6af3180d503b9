// The 3D right-hand side with its tiles staged by the tensor memory accelerator (TMA): same decomposition and the same
// per-plane schedule as rhs_fused_march_kernel (mfc_fused.cuh: tile in (x, y), march along z three planes ahead, z window
// in tensor memory), but every global read of q is a cp.async.bulk.tensor box issued by ONE thread and completed on an
// mbarrier (UTMALDG in the SASS), instead of ~20 eight-byte cp.async per thread and plane with their index arithmetic:
//   * the ghost cells of q are filled IN MEMORY before the launch (ghost_fill_kernel), so a tile's halo is a
//     plain box of the padded array whatever the boundary kind -- no wrapped / clamped index map in the kernel;
//   * plane ip + 1 WITH its halo (38 x (TY + 6) cells x NEQ) lands in the staged-plane buffer P[(ip + 1) & 1] directly
//     (P is double-buffered); its halo cells are converted to primitives in place, its own cells are overwritten with the
//     primitives kept in the TMEM ring -- no separate halo buffers, no halo copy;
//   * the raw own column of plane m + 1 (32 x TY x NEQ) lands in SQ and is converted straight into the TMEM ring; the
//     raw q_s of the cell being written lands in SS (same box of the same array: q_s is the array L is evaluated on).
// A TMA box must START at a 16-byte aligned global address (measured: an odd x origin of a box of doubles raises an
// illegal-instruction fault), so rows must be 16-byte aligned -- even padded extent in x and a 16-byte aligned base;
// otherwise the launcher uses rhs_fused_march_kernel -- and box origins in x must be even: the staged plane starts at
// padded x = x0 (even), the own-column boxes start one cell early (padded x0 + 2) and are FTX + 2 wide.  Boxes that stick out of the padded array (ragged last tiles) are zero-filled by the TMA; those
// cells belong to threads that write nothing and feed no active cell.
#pragma once
#include <cuda.h>

#include "mfc_fused.cuh"

namespace mfc {

__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MFC_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MFC_DONE;\n"
        "bra MFC_WAIT;\n"
        "MFC_DONE:\n"
        "}\n" ::"r"(smem_addr(bar)), "r"(parity)
        : "memory");
}
// one box of the rank-4 tensor (x, y, z, equation) -> dense shared memory [equation][z][y][x]
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, unsigned long long *bar, int cx, int cy, int cz, int ce)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(
            smem_addr(dst)),
        "l"(reinterpret_cast<unsigned long long>(map)), "r"(smem_addr(bar)), "r"(cx), "r"(cy), "r"(cz), "r"(ce)
        : "memory");
}

template <int NF, int TY>
struct TmaCfg {
    using C = FusedCfg<3, NF, TY>;
    static constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL;
    static constexpr int CW = FTX + 2;                                   // row length of an own-column box: cells -1 .. FTX
    static constexpr int NB = TY * CW;                                   // cells per variable of an own-column box
    static constexpr int r16(int v) { return (v + 15) / 16 * 16; }       // 128-byte granules, in doubles
    static constexpr int nPb = r16(NEQ * PPL);                           // one staged plane
    static constexpr int oRim = 2 * nPb;
    static constexpr int oX8 = oRim + C::nHx + C::nHy;
    static constexpr int oX = oX8 + NT;
    static constexpr int oX2 = oX + NEQ * NT;
    static constexpr int oSQ = r16(oX2 + NEQ * NT);
    static constexpr int oSS = oSQ + r16(NEQ * NB);
    static constexpr int oBar = oSS + r16(NEQ * NB);                     // FULL_P[2], FULL_SQ, FULL_SS, TMEM base word
    static constexpr int doubles = oBar + 8;
    static constexpr int bytes = doubles * (int)sizeof(double);
    static constexpr unsigned plane_bytes = NEQ * PPL * sizeof(double);
    static constexpr unsigned col_bytes = NEQ * NB * sizeof(double);
    // one block per multiprocessor is what the TMEM allocation (all 512 columns) relies on
    static_assert(2 * bytes > 227 * 1024, "two resident blocks would deadlock in tcgen05.alloc");
};

template <int NF, int TY, int ORDER, bool NU>
__global__ void __launch_bounds__(FTX *TY, 1)
    rhs_fused_march_tma_kernel(const __grid_constant__ CUtensorMap tm_plane, const __grid_constant__ CUtensorMap tm_col, typename GeoOf<NU>::type g, Eos eos,
                               SweepOut o, int ntx, int nty, int seg)
{
    constexpr int D = 3;
    using C = FusedCfg<D, NF, TY>;
    using T = TmaCfg<NF, TY>;
    using I = Idx<D, NF>;
    constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, NH = C::NH, NHT = C::NHT;
    extern __shared__ __align__(128) double sm[];
    double *const rim = sm + T::oRim;
    double *const X8 = sm + T::oX8;
    double *const X = sm + T::oX;                                   // [NEQ][NT]  y exchange, right states
    double *const X2 = sm + T::oX2;                                 // [NEQ][NT]  y exchange, fluxes
    double *const SQ = sm + T::oSQ;                                 // [NEQ][TY][CW]  raw q, own column, next plane
    double *const SS = sm + T::oSS;                                 // [NEQ][TY][CW]  raw q_s of the cell being written
    unsigned long long *const bars = reinterpret_cast<unsigned long long *>(sm + T::oBar);
    unsigned long long *const FULL_P = bars;                        // [2]
    unsigned long long *const FULL_SQ = bars + 2;
    unsigned long long *const FULL_SS = bars + 3;
    unsigned *const tmem_word = reinterpret_cast<unsigned *>(bars + 4);
    constexpr int TV = NEQ + 1 <= 8 ? 8 : 10;
    enum { T_RING = 0, T_PARK = 4, T_PREV = 5, T_FLUX = 6, T_SLOTS = 7 };
    static_assert(T_SLOTS * 2 * TV * ((TY + 3) / 4) <= 512, "TMEM columns");

    const int tid = threadIdx.x, i = tid & 31, j = tid >> 5;
    int b = blockIdx.x;
    const int bx = b % ntx;
    b /= ntx;
    const int by = b % nty, bs = b / nty;
    const int x0 = bx * FTX, y0 = by * TY;
    const int k0 = bs * seg, k1 = min(k0 + seg, g.n[2]);
    const bool active = x0 + i < g.n[0] && y0 + j < g.n[1];
    const long long col = (long long)(y0 + j + NG) * g.sy + (x0 + i + NG);
    constexpr int POWN = NG * FPX + NG;                             // own cell (0, 0) of a staged plane
    const int pown = POWN + j * FPX + i;
    constexpr int NB = T::NB;
    const int bown = j * T::CW + i + 1;                             // own cell in an own-column box
    // halo cells of this thread: position in the staged plane (row-major numbering that skips the interior block)
    int hpos[NHT];
#pragma unroll
    for (int t = 0; t < NHT; ++t) {
        const int h = tid + t * NT;
        constexpr int TOP = NG * FPX;
        int c = 0;
        if (h < TOP) c = h;
        else if (h < TOP + 2 * NG * TY) {
            const int r = (h - TOP) / (2 * NG), k = (h - TOP) - r * 2 * NG;
            c = (NG + r) * FPX + (k < NG ? k : FTX + k);
        } else if (h < NH) c = (NG + TY) * FPX + (h - TOP - 2 * NG * TY);
        hpos[t] = c;
    }

    if (tid == 0) {
        mbar_init(FULL_P, 1);
        mbar_init(FULL_P + 1, 1);
        mbar_init(FULL_SQ, 1);
        mbar_init(FULL_SS, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (j == 0) tmem_alloc512(tmem_word);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem_base = *tmem_word;
    const unsigned tbase = tmem_base + ((unsigned)(32 * (j & 3)) << 16) + (unsigned)((j >> 2) * T_SLOTS * 2 * TV);
    auto tslot = [&](int s) -> unsigned { return tbase + (unsigned)(s * 2 * TV); };
    {
        double z[TV];
#pragma unroll
        for (int k = 0; k < TV; ++k) z[k] = 0.0;
        tmem_store<TV>(tslot(T_FLUX), z);
        tmem_store<TV>(tslot(T_PREV), z);
    }

    // raw column of plane m (landed in SQ) -> primitives -> ring slot of plane m (that of plane m - 4, dead by now)
    auto convert_column = [&](int m) {
        double qc[NEQ], wc[TV];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) qc[e] = SQ[e * NB + bown];
        {
            double w7[NEQ];
            cons_to_prim_cell<D, NF>(qc, eos, w7);
#pragma unroll
            for (int e = 0; e < NEQ; ++e) wc[e] = w7[e];
#pragma unroll
            for (int k = NEQ; k < TV; ++k) wc[k] = 0.0;
        }
        tmem_store<TV>(tslot(T_RING + (m & 3)), wc);
    };

    // Iteration m (ip = m - 3), cf. mfc_fused.cuh:
    //   top      thread 0 issues {plane ip + 1 with halo -> P[(ip + 1) & 1]} and {q_s of plane ip -> SS}
    //   in-plane x and y differences of plane ip from P[ip & 1]; behind its first barrier column m (SQ) is converted
    //            into the ring; behind its second barrier thread 0 issues {column m + 1 -> SQ}
    //   bottom   z part of cell ip (window from the ring), output;  glue: halo cells of P[(ip + 1) & 1] converted in
    //            place, its own cells taken from the ring
    //   barrier  (every buffer the next issues overwrite has been read)
    const int pstart = k0 - NG, pend = k1 + NG;
    if (tid == 0) {
        mbar_expect_tx(FULL_SQ, T::col_bytes);
        tma_load_4d(SQ, &tm_col, FULL_SQ, x0 + NG - 1, y0 + NG, pstart + NG, 0);
    }
#pragma unroll 1
    for (int m = pstart; m < pend; ++m) {
        const int n = m - pstart;
        const int ip = m - NG;
        const bool inplane = ip >= k0;
        const bool next_inplane = ip + 1 >= k0 && ip + 1 < k1;
        const long long cell = (long long)(ip + NG) * g.sz + col;
        double *const Pcur = sm + (ip & 1) * T::nPb;                // meaningful when inplane
        double *const Pnext = sm + ((ip + 1) & 1) * T::nPb;
        double coef = o.coef;
        asm volatile("" : "+d"(coef));
        NuPlane nup{nullptr, nullptr, 0, 0};
        if constexpr (NU) nup = NuPlane{g.nu[0] + x0 + NG, g.nu[1] + y0 + NG, g.nus[0], g.nus[1]};
        double cx, cy, cz;
        if constexpr (NU) {                                         // the cell's own widths (Eq. 8-9)
            cx = coef * __ldg(nup.tx + i + 27 * nup.sx);
            cy = coef * __ldg(nup.ty + j + 27 * nup.sy);
            cz = coef * __ldg(g.nu[2] + max(ip, 0) + NG + 27 * g.nus[2]);
        } else {
            cx = coef * g.inv_dx[0], cy = coef * g.inv_dx[1], cz = coef * g.inv_dx[2];
        }

        if (tid == 0) {
            if (next_inplane) {
                mbar_expect_tx(FULL_P + ((ip + 1) & 1), T::plane_bytes);
                tma_load_4d(Pnext, &tm_plane, FULL_P + ((ip + 1) & 1), x0, y0, ip + 1 + NG, 0);
            }
            if (inplane && o.nbase > 0) {
                mbar_expect_tx(FULL_SS, T::col_bytes);
                tma_load_4d(SS, &tm_col, FULL_SS, x0 + NG - 1, y0 + NG, ip + NG, 0);
            }
        }

        double acc[NEQ];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) acc[e] = 0.0;
        if (inplane) {
            auto early = [&]() {
                if (active && o.nbase > 1 && ip + 1 < k1) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) prefetch_l2(o.qn + (long long)e * g.cells + cell + g.sz);
                }
            };
            auto mid = [&]() {
                mbar_wait(FULL_SQ, n & 1);
                convert_column(m);
            };
            const InplaneBufs<D, NF, TY> B(Pcur, rim, X, X2, X8);
            inplane_xy<D, NF, TY, ORDER, NU>(B, eos, cx, cy, acc, early, mid, nup);
        } else {
            mbar_wait(FULL_SQ, n & 1);
            convert_column(m);
            __syncthreads();                                        // SQ has been read by everybody
        }
        if (tid == 0 && m + 1 < pend) {                             // behind a barrier that follows the last read of SQ
            mbar_expect_tx(FULL_SQ, T::col_bytes);
            tma_load_4d(SQ, &tm_col, FULL_SQ, x0 + NG - 1, y0 + NG, m + 1 + NG, 0);
        }

        // ---- bottom of the iteration ----
        double qnv[NEQ];
        if (inplane) {
            if (active && o.nbase > 1) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e) qnv[e] = __ldcg(o.qn + (long long)e * g.cells + cell);
            }
            if (o.nbase > 0) {
                mbar_wait(FULL_SS, (ip - k0) & 1);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) acc[e] = fma(o.cb, SS[e * NB + bown], acc[e]);
            }
        }
        double wn[TV], vb[TV];
        tmem_load<TV>(tslot(T_RING + (m & 3)), wn);                 // plane m, converted above
        if (inplane) {
#pragma unroll
            for (int k = NEQ; k < TV; ++k) vb[k] = 0.0;
#pragma unroll
            for (int e = 0; e < NEQ; ++e) vb[e] = Pcur[e * PPL + pown];
        } else if (n >= 3) {
            tmem_load<TV>(tslot(T_RING + ((m + 1) & 3)), vb);
        } else {
#pragma unroll
            for (int k = 0; k < TV; ++k) vb[k] = 0.0;
        }
        auto glue = [&]() {
            if (next_inplane) {
                mbar_wait(FULL_P + ((ip + 1) & 1), ((ip + 1 - k0) >> 1) & 1);
#pragma unroll
                for (int t = 0; t < NHT; ++t) {
                    if (tid + t * NT < NH) {
                        double qc[NEQ], wc[NEQ];
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) qc[e] = Pnext[e * PPL + hpos[t]];
                        cons_to_prim_cell<D, NF>(qc, eos, wc);
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) Pnext[e * PPL + hpos[t]] = wc[e];
                    }
                }
                double rp[TV];                                      // plane m - 2 = ip + 1
                tmem_load<TV>(tslot(T_RING + ((m + 2) & 3)), rp);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) Pnext[e * PPL + pown] = rp[e];
            }
        };
        auto zpart = [&]() {
            if (n >= 4) {
                const int c = m - 2;
                double rc[TV], rd[TV], vLp[TV], vprev[TV], vL[TV], vR[NEQ];
                tmem_load<TV>(tslot(T_RING + ((m + 2) & 3)), rc);   // plane m - 2
                tmem_load<TV>(tslot(T_RING + ((m + 3) & 3)), rd);   // plane m - 1
                tmem_load<TV>(tslot(T_PARK), vLp);
                tmem_load<TV>(tslot(T_PREV), vprev);
#pragma unroll
                for (int k = NEQ; k < TV; ++k) vL[k] = 0.0;
                NuRef nz{nullptr, 0};
                if constexpr (NU) nz = NuRef{g.nu[2] + c + NG, g.nus[2]};
#pragma unroll
                for (int e = 0; e < NEQ; ++e)
                    reconstruct<ORDER, NU>(rc[e], vb[e] - vprev[e], rc[e] - vb[e], rd[e] - rc[e], wn[e] - rd[e], eos.weno_eps4, vL[e], vR[e], nz);
                tmem_store<TV>(tslot(T_PARK), vL);
                if (c >= k0) {
                    double Fm[TV], Fn[TV];
                    tmem_load<TV>(tslot(T_FLUX), Fm);
                    double Fp[NEQ], ufp, vl7[NEQ];
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) vl7[e] = vLp[e];
                    hllc<D, NF, 2>(vl7, vR, eos, Fp, ufp);
                    const double du = ufp - Fm[NEQ];
#pragma unroll
                    for (int k = 0; k < TV; ++k) Fn[k] = 0.0;
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) {
                        double rr = Fm[e] - Fp[e];
                        if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, vb[e], vb[I::E]), du, rr);
                        acc[e] = fma(cz, rr, acc[e]);
                        Fn[e] = Fp[e];
                    }
                    Fn[NEQ] = ufp;
                    tmem_store<TV>(tslot(T_FLUX), Fn);
                }
            }
            tmem_store<TV>(tslot(T_PREV), vb);
            if (inplane && active) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e)
                    o.out[(long long)e * g.cells + cell] = o.nbase > 1 ? fma(o.ca, qnv[e], acc[e]) : acc[e];
            }
        };
        if ((j >> 2) & 1) {
            glue();
            zpart();
        } else {
            zpart();
            glue();
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); // this thread's writes to P / reads of SS before the next boxes
        __syncthreads();
    }
    if (j == 0) tmem_dealloc512(tmem_base);
}

}  // namespace mfc
