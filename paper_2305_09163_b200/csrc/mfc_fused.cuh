// The whole right-hand side L(q) in ONE kernel: ghost fill + cons->prim at load (a0, a1), WENO5 + HLLC in
// x, y and z (a2, a3), flux difference + alpha div u (a4) and the Runge-Kutta stage combine (a5).
//
// Why one kernel.  The path is bound by the FP64 pipe (about 1600 DADD/DMUL/DFMA per cell and evaluation
// against 160 B of compulsory traffic), so every byte that a per-direction design moves
// more than once (primitive array, partial RHS) is time taken from an already memory-heavy schedule.  Here a
// cell of q is read once from HBM (plus halo re-reads that hit L2) and a cell of the result is written once.
//
// Decomposition.  A block owns a tile of FTX x TY cells in (x, y) and MARCHES along z over a segment of the
// domain; thread (i, j) = (lane, warp) owns the column (x0 + i, y0 + j).
//   * every plane is loaded once, with a halo of 3 cells in x and y, converted to primitives on the way
//     (ghost cells take the wrapped / clamped interior cell) and kept in shared memory (P);
//   * x: each thread reconstructs its own cell from P; right states and fluxes move between neighbouring
//     lanes by warp shuffles (tile width = warp width);
//   * y: same, the exchange between neighbouring warps goes through shared memory (X);
//   * z: the 5-plane window of a column is thread-private: four older planes in a shared-memory ring (R) plus
//     the plane in P; the left state of the previous face is parked in shared memory, the previous flux stays
//     in registers, so every cell is reconstructed once and every face solved once along the march;
//   * the rim of the tile (left state of face -1/2 from cell -1, right state of the face past the last cell,
//     in x and in y) is reconstructed by the first three warps while the others start on the z direction; the
//     rim faces themselves are solved by one warp each once the first row / lane has published its state;
//   * the in-plane part of cell (., ., p), ca q_n + coef (L_x + L_y), is written when plane p is loaded; the z
//     part and cb q_s are added three planes later, when face p + 1/2 is known (the line is still in L2; the
//     loads are issued before the Riemann solve that produces the last term, so their latency is covered).
// FP64 issue needs instruction-level parallelism rather than many warps on this part (one warp per scheduler
// with four independent chains already reaches 92 % of the DFMA peak), so the block is 16 warps with up to
// 128 registers each and the seven variables are reconstructed as independent chains.
#pragma once
#include "mfc_math.cuh"

namespace mfc {

constexpr int FTX = 32;             // tile width in x = warp width
constexpr int FPX = FTX + 2 * NG;   // staged row length

template <int D, int NF, int TY>
struct FusedCfg {
    static constexpr int NEQ = 2 * NF + D;
    static constexpr int HY = D >= 2 ? NG : 0;
    static constexpr int PY = TY + 2 * HY;
    static constexpr int NT = FTX * TY;
    static constexpr int PPL = PY * FPX;                            // doubles per variable in the staged plane
    static constexpr int nP = NEQ * PPL;
    static constexpr int nX = D >= 2 ? (NEQ + 1) * NT : 0;          // y exchange: right states, then fluxes
    // rim of the tile in x, per row: vL of cell -1, vR of cell 0, vR of cell FTX, flux of lane 0; the rim flux
    // overwrites the first two once they have been read (by the thread that writes it)
    static constexpr int nHx = (3 * NEQ + (NEQ + 1)) * TY;
    // rim in y, per column: vL of row -1, vR of row TY; the rim flux overwrites them likewise
    static constexpr int nHy = D >= 2 ? 2 * NEQ * FTX : 0;
    static constexpr int nR = D == 3 ? 5 * NEQ * NT : 0;            // four ring slots + parked left state
    static constexpr int doubles = nP + nX + nHx + nHy + nR;
    static constexpr int bytes = doubles * (int)sizeof(double);
    static_assert(TY <= 16, "the x rim jobs are laid out for at most 16 rows");
};

__device__ __forceinline__ void prefetch_l2(const double *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

template <int D, int NF, int TY>
__global__ void __launch_bounds__(FTX *TY, 1)
    rhs_fused_kernel(Geo g, Eos eos, const double *__restrict__ q, SweepOut o, int ntx, int nty, int seg)
{
    using C = FusedCfg<D, NF, TY>;
    using I = Idx<D, NF>;
    constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, HY = C::HY;
    constexpr int NA1 = I::NA > 0 ? I::NA : 1;
    constexpr int RIMW = TY - 1;                                    // warp that solves the rim faces
    extern __shared__ double sm[];
    double *const P = sm;
    double *const X = P + C::nP;
    double *const HxL = X + C::nX;                                  // [NEQ][TY]   left state of face -1/2
    double *const ExR = HxL + NEQ * TY;                             // [NEQ][TY]   right state of face -1/2 (lane 0)
    double *const HxR = ExR + NEQ * TY;                             // [NEQ][TY]   right state of face FTX - 1/2
    double *const ExF = HxR + NEQ * TY;                             // [NEQ+1][TY] flux of face 1/2 (lane 0)
    double *const FxH = HxL;                                        // [NEQ+1][TY] flux of face -1/2: over HxL, ExR[0]
    double *const HyL = ExF + (NEQ + 1) * TY;                       // [NEQ][FTX]
    double *const HyR = HyL + (D >= 2 ? NEQ * FTX : 0);             // [NEQ][FTX]
    double *const FyH = HyL;                                        // [NEQ+1][FTX] over HyL, HyR[0]
    double *const R = HyR + (D >= 2 ? NEQ * FTX : 0);
    double *const park = R + (D == 3 ? 4 * NEQ * NT : 0);

    const int tid = threadIdx.x, i = tid & 31, j = tid >> 5;
    int b = blockIdx.x;
    const int bx = b % ntx;
    b /= ntx;
    const int by = b % nty, bs = b / nty;
    const int x0 = bx * FTX, y0 = by * TY;
    const int k0 = D == 3 ? bs * seg : 0;
    const int k1 = D == 3 ? min(k0 + seg, g.n[2]) : 1;
    const bool active = x0 + i < g.n[0] && (D < 2 || y0 + j < g.n[1]);
    const long long col = (long long)(x0 + i + NG) + (D >= 2 ? (long long)(y0 + j + NG) * g.sy : 0);
    const double *const pc = P + (j + HY) * FPX + (i + NG);         // this thread's cell in the staged plane
    const double cx = o.coef * g.inv_dx[0], cy = D >= 2 ? o.coef * g.inv_dx[1] : 0.0, cz = D == 3 ? o.coef * g.inv_dx[2] : 0.0;

    // source cell of staged position c of plane p (ghost fill = index map)
    auto source = [&](int p, int c) -> long long {
        const int jj = c / FPX, ii = c - jj * FPX;
        long long src = bc_source(min(x0 - NG + ii, g.n[0] + NG - 1), g.n[0], g.bc_lo[0], g.bc_hi[0]) + NG;
        if (D >= 2) src += (long long)(bc_source(min(y0 - NG + jj, g.n[1] + NG - 1), g.n[1], g.bc_lo[1], g.bc_hi[1]) + NG) * g.sy;
        if (D == 3) src += (long long)(bc_source(min(max(p, -NG), g.n[2] + NG - 1), g.n[2], g.bc_lo[2], g.bc_hi[2]) + NG) * g.sz;
        return src;
    };
    constexpr int NIT = (C::PY * FPX + NT - 1) / NT;
    auto load_plane = [&](int p) {                                  // every load is issued before the first conversion
        double qc[NIT][NEQ];
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int c = tid + it * NT;
            if (c < C::PY * FPX) {
                const long long src = source(p, c);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) qc[it][e] = __ldg(q + (long long)e * g.cells + src);
            }
        }
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int c = tid + it * NT;
            if (c < C::PY * FPX) {
                double wc[NEQ];
                cons_to_prim_cell<D, NF>(qc[it], eos, wc);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) P[e * PPL + c] = wc[e];
            }
        }
    };
    auto prefetch_plane = [&](int p) {
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int c = tid + it * NT;
            if (c < C::PY * FPX) {
                const long long src = source(p, c);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) prefetch_l2(q + (long long)e * g.cells + src);
            }
        }
    };

    double Fmz[NEQ], ufmz = 0.0;                                    // flux and face velocity of the previous z face
#pragma unroll
    for (int e = 0; e < NEQ; ++e) Fmz[e] = 0.0;

    const int pstart = D == 3 ? k0 - NG : 0, pend = D == 3 ? k1 + NG : 1;
    load_plane(pstart);
    __syncthreads();
#pragma unroll 1
    for (int p = pstart; p < pend; ++p) {
        const int n = p - pstart;                                   // planes loaded before this one
        if (D == 3 && p + 1 < pend) {
            prefetch_plane(p + 1);
            // q_n of the cell whose in-plane part the next iteration writes
            if (o.nbase > 1 && active && p + 1 >= k0 && p + 1 < k1) {
                const double *pq = o.qn + (long long)(p + 1 + NG) * g.sz + col;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) prefetch_l2(pq + (long long)e * g.cells);
            }
        }

        // ---- z: reconstruct cell p - 2, solve face (p - 2) - 1/2, close cell p - 3 ----
        if constexpr (D == 3) if (n >= 4) {
            const int c = p - 2;
            const bool close = c > k0 && active;
            const double *const ra = R + ((n + 0) & 3) * NEQ * NT + tid;
            const double *const rb = R + ((n + 1) & 3) * NEQ * NT + tid;
            const double *const rc = R + ((n + 2) & 3) * NEQ * NT + tid;
            const double *const rd = R + ((n + 3) & 3) * NEQ * NT + tid;
            double vLp[NEQ], vL[NEQ], vR[NEQ], ab[NA1];
#pragma unroll
            for (int e = 0; e < NEQ; ++e) vLp[e] = park[e * NT + tid];
#pragma unroll
            for (int e = 0; e < NEQ; ++e) {
                const double va = ra[e * NT], vb = rb[e * NT], vc = rc[e * NT], vd = rd[e * NT], ve = pc[e * PPL];
                weno5(vc, vb - va, vc - vb, vd - vc, ve - vd, eos.weno_eps4, vL[e], vR[e]);
                if (e >= I::A) ab[e - I::A] = vb;
            }
#pragma unroll
            for (int e = 0; e < NEQ; ++e) park[e * NT + tid] = vL[e];
            if (c >= k0) {
                // partial result and q_s term of the cell about to be closed: issued before the Riemann solve
                const long long cell = (long long)(c - 1 + NG) * g.sz + col;
                double ob[NEQ];
                if (close) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) {
                        ob[e] = o.out[(long long)e * g.cells + cell];
                        if (o.nbase > 0) ob[e] = fma(o.cb, __ldg(o.qs + (long long)e * g.cells + cell), ob[e]);
                    }
                }
                double Fp[NEQ], ufp;
                hllc<D, NF, 2>(vLp, vR, eos, Fp, ufp);
                if (close) {
                    const double du = ufp - ufmz;
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) {
                        double rr = Fmz[e] - Fp[e];
                        if (e >= I::A) rr = fma(ab[e - I::A], du, rr);
                        o.out[(long long)e * g.cells + cell] = fma(cz, rr, ob[e]);
                    }
                }
#pragma unroll
                for (int e = 0; e < NEQ; ++e) Fmz[e] = Fp[e];
                ufmz = ufp;
            }
        }

        const bool inplane = D < 3 || (p >= k0 && p < k1);          // block-uniform
        if (inplane) {
            // ---- rim states: left state of face -1/2 (from cell -1) and right state of the face past the tile ----
            for (int job = tid; job < (D >= 2 ? 96 : 32); job += NT) {
                const bool inx = job < 32;
                const int r = inx ? (job & 15) : (job & 31);
                const bool left = inx ? job < 16 : job < 64;
                if (!inx || r < TY) {
                    // centre cell of the reconstruction: -1 (left) or T (right) along the normal direction
                    const int st = inx ? 1 : FPX;
                    const double *pb = inx ? P + (r + HY) * FPX + NG + (left ? -1 : FTX) : P + (HY + (left ? -1 : TY)) * FPX + NG + r;
                    double *dst = inx ? (left ? HxL : HxR) + r : (left ? HyL : HyR) + r;
                    const int ds = inx ? TY : FTX;
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) {
                        const double *s5 = pb + e * PPL;
                        double vl, vr;
                        weno5(s5[0], s5[-st] - s5[-2 * st], s5[0] - s5[-st], s5[st] - s5[0], s5[2 * st] - s5[st], eos.weno_eps4, vl, vr);
                        dst[e * ds] = left ? vl : vr;
                    }
                }
            }

            // ---- y, first half: reconstruct, publish the right state ----
            double vLy[NEQ];
            if constexpr (D >= 2) {
                double vRy[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double *s5 = pc + e * PPL;
                    weno5(s5[0], s5[-FPX] - s5[-2 * FPX], s5[0] - s5[-FPX], s5[FPX] - s5[0], s5[2 * FPX] - s5[FPX], eos.weno_eps4, vLy[e], vRy[e]);
                }
#pragma unroll
                for (int e = 0; e < NEQ; ++e) X[e * NT + tid] = vRy[e];
            }
            __syncthreads();                                        // S1: rim states and y right states are visible

            // ---- x: reconstruct, exchange by shuffles, solve face i + 1/2, difference ----
            double acc[NEQ];
            {
                double vL[NEQ], vR[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double *s5 = pc + e * PPL;
                    weno5(s5[0], s5[-1] - s5[-2], s5[0] - s5[-1], s5[1] - s5[0], s5[2] - s5[1], eos.weno_eps4, vL[e], vR[e]);
                }
                if (i == 0) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) ExR[e * TY + j] = vR[e];
                }
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double nb = __shfl_down_sync(0xffffffffu, vR[e], 1);
                    vR[e] = i == FTX - 1 ? HxR[e * TY + j] : nb;
                }
                double Fp[NEQ], ufp;
                hllc<D, NF, 0>(vL, vR, eos, Fp, ufp);
                if (i == 0) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) ExF[e * TY + j] = Fp[e];
                    ExF[NEQ * TY + j] = ufp;
                }
                const double du = ufp - __shfl_up_sync(0xffffffffu, ufp, 1);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double rr = __shfl_up_sync(0xffffffffu, Fp[e], 1) - Fp[e];
                    if (e >= I::A) rr = fma(pc[e * PPL], du, rr);
                    acc[e] = cx * rr;                               // lane 0 is redone below with the rim flux
                }
            }

            // ---- y, second half: solve face j + 1/2 (and, one warp, the rim faces j = -1/2) ----
            double Fy[NEQ > 0 ? NEQ : 1], ufy = 0.0;
            if constexpr (D >= 2) {
                double vRn[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) vRn[e] = j == TY - 1 ? HyR[e * FTX + i] : X[e * NT + tid + FTX];
                hllc<D, NF, 1>(vLy, vRn, eos, Fy, ufy);
                if (j == RIMW) {
                    double hl[NEQ], hr[NEQ], F[NEQ], uf;
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) { hl[e] = HyL[e * FTX + i]; hr[e] = X[e * NT + i]; }
                    hllc<D, NF, 1>(hl, hr, eos, F, uf);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) FyH[e * FTX + i] = F[e];
                    FyH[NEQ * FTX + i] = uf;
                }
            }
            __syncthreads();                                        // S2: y right states have been read, lane-0 states are visible
            if constexpr (D >= 2) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e) X[e * NT + tid] = Fy[e];
                X[NEQ * NT + tid] = ufy;
            }
            if (j == RIMW && i < TY) {                              // rim faces i = -1/2, one per row
                double hl[NEQ], hr[NEQ], F[NEQ], uf;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) { hl[e] = HxL[e * TY + i]; hr[e] = ExR[e * TY + i]; }
                hllc<D, NF, 0>(hl, hr, eos, F, uf);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) FxH[e * TY + i] = F[e];
                FxH[NEQ * TY + i] = uf;
            }
            __syncthreads();                                        // S3: fluxes are visible
            if (i == 0) {
                const double du = ExF[NEQ * TY + j] - FxH[NEQ * TY + j];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double rr = FxH[e * TY + j] - ExF[e * TY + j];
                    if (e >= I::A) rr = fma(pc[e * PPL], du, rr);
                    acc[e] = cx * rr;
                }
            }
            if constexpr (D >= 2) {
                const double ufm = j == 0 ? FyH[NEQ * FTX + i] : X[NEQ * NT + tid - FTX];
                const double du = ufy - ufm;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double fm = j == 0 ? FyH[e * FTX + i] : X[e * NT + tid - FTX];
                    double rr = fm - Fy[e];
                    if (e >= I::A) rr = fma(pc[e * PPL], du, rr);
                    acc[e] = fma(cy, rr, acc[e]);
                }
            }

            // ---- a4 + a5: coef (L_x + L_y) + ca q_n now (out may be q_n itself, so q_n is read before this cell of
            // out is first written); the z part and cb q_s follow three planes later ----
            if (active) {
                const long long cell = (D == 3 ? (long long)(p + NG) * g.sz : 0) + col;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double v = acc[e];
                    if (o.nbase > 1) v = fma(o.ca, o.qn[(long long)e * g.cells + cell], v);
                    if (D < 3 && o.nbase > 0) v = fma(o.cb, o.qs[(long long)e * g.cells + cell], v);
                    o.out[(long long)e * g.cells + cell] = v;
                }
            }
        }

        if constexpr (D == 3) {
            // the plane enters the ring (slot of the plane that just left the window), then the next one is staged
            double *const rs = R + (n & 3) * NEQ * NT + tid;
#pragma unroll
            for (int e = 0; e < NEQ; ++e) rs[e * NT] = pc[e * PPL];
            if (p + 1 < pend) {
                __syncthreads();                                    // S4: P is free
                load_plane(p + 1);
                __syncthreads();                                    // S0
            }
        }
    }
}

}  // namespace mfc
