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
//   * the faces on the rim of the tile (x: -1/2 and right state of cell FTX; y likewise) are "halo jobs"
//     done by the first three warps while the others start on the z direction;
//   * the in-plane part of cell (., ., p) is written as out = base + coef (L_x + L_y) when plane p is loaded;
//     the z part is added three planes later, when face p + 1/2 is known (the line is still in L2).
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
    static constexpr int nHx = (2 * NEQ + 1) * TY;                  // rim of the tile in x: vR[NEQ][TY], F[NEQ+1][TY]
    static constexpr int nHy = D >= 2 ? (2 * NEQ + 1) * FTX : 0;    // rim in y
    static constexpr int nR = D == 3 ? 5 * NEQ * NT : 0;            // four ring slots + parked left state
    static constexpr int doubles = nP + nX + nHx + nHy + nR;
    static constexpr int bytes = doubles * (int)sizeof(double);
    static_assert(TY <= 16, "the x rim jobs are laid out for at most 16 rows");
};

__device__ __forceinline__ void prefetch_l2(const double *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// left state of the face below cell 0 (seen from cell -1) and right state of the same face (seen from cell 0);
// pb points at cell 0 of variable 0, st is the stride along the normal direction
template <int NEQ>
__device__ __forceinline__ void rim_face_states(const double *pb, int st, int ppl, double eps4, double (&vL)[NEQ], double (&vR)[NEQ])
{
#pragma unroll
    for (int e = 0; e < NEQ; ++e) {
        const double *p = pb + e * ppl;
        const double a = p[-3 * st], b = p[-2 * st], c = p[-st], d = p[0], f = p[st], h = p[2 * st];
        double unused;
        weno5(c, b - a, c - b, d - c, f - d, eps4, vL[e], unused);
        weno5(d, c - b, d - c, f - d, h - f, eps4, unused, vR[e]);
    }
}

template <int D, int NF, int TY>
__global__ void __launch_bounds__(FTX *TY, 1)
    rhs_fused_kernel(Geo g, Eos eos, const double *__restrict__ q, SweepOut o, int ntx, int nty, int seg)
{
    using C = FusedCfg<D, NF, TY>;
    using I = Idx<D, NF>;
    constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, HY = C::HY;
    constexpr int NA1 = I::NA > 0 ? I::NA : 1;
    extern __shared__ double sm[];
    double *const P = sm;
    double *const X = P + C::nP;
    double *const HxR = X + C::nX;
    double *const FxH = HxR + NEQ * TY;
    double *const HyR = FxH + (NEQ + 1) * TY;
    double *const FyH = HyR + (D >= 2 ? NEQ * FTX : 0);
    double *const R = FyH + (D >= 2 ? (NEQ + 1) * FTX : 0);
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
    auto load_plane = [&](int p) {
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int c = tid + it * NT;
            if (c < C::PY * FPX) {
                const long long src = source(p, c);
                double qc[NEQ], wc[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) qc[e] = __ldg(q + (long long)e * g.cells + src);
                cons_to_prim_cell<D, NF>(qc, eos, wc);
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
        if (D == 3 && p + 1 < pend) prefetch_plane(p + 1);

        // ---- z: reconstruct cell p - 2, solve face (p - 2) - 1/2, close cell p - 3 ----
        if constexpr (D == 3) if (n >= 4) {
            const int c = p - 2;
            const bool close = c > k0 && active;
            double *const op = o.out + (long long)(c - 1 + NG) * g.sz + col;
            double ob[NEQ];
            if (close) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e) ob[e] = op[(long long)e * g.cells];
            }
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
                double Fp[NEQ], ufp;
                hllc<D, NF, 2>(vLp, vR, eos, Fp, ufp);
                if (close) {
                    const double du = ufp - ufmz;
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) {
                        double rr = Fmz[e] - Fp[e];
                        if (e >= I::A) rr = fma(ab[e - I::A], du, rr);
                        op[(long long)e * g.cells] = fma(cz, rr, ob[e]);
                    }
                }
#pragma unroll
                for (int e = 0; e < NEQ; ++e) Fmz[e] = Fp[e];
                ufmz = ufp;
            }
        }

        const bool inplane = D < 3 || (p >= k0 && p < k1);          // block-uniform
        if (inplane) {
            // ---- rim of the tile: faces -1/2 and right states of the cell past the last one ----
            for (int job = tid; job < (D >= 2 ? 96 : 32); job += NT) {
                if (job < 16) {
                    if (job < TY) {
                        double vL[NEQ], vR[NEQ], F[NEQ], uf;
                        rim_face_states<NEQ>(P + (job + HY) * FPX + NG, 1, PPL, eos.weno_eps4, vL, vR);
                        hllc<D, NF, 0>(vL, vR, eos, F, uf);
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) FxH[e * TY + job] = F[e];
                        FxH[NEQ * TY + job] = uf;
                    }
                } else if (job < 32) {
                    const int r = job - 16;
                    if (r < TY) {
                        const double *pb = P + (r + HY) * FPX + NG + FTX;
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) {
                            const double *s = pb + e * PPL;
                            double unused, v;
                            weno5(s[0], s[-1] - s[-2], s[0] - s[-1], s[1] - s[0], s[2] - s[1], eos.weno_eps4, unused, v);
                            HxR[e * TY + r] = v;
                        }
                    }
                } else if constexpr (D >= 2) { if (job < 64) {
                    const int cc = job - 32;
                    double vL[NEQ], vR[NEQ], F[NEQ], uf;
                    rim_face_states<NEQ>(P + HY * FPX + NG + cc, FPX, PPL, eos.weno_eps4, vL, vR);
                    hllc<D, NF, 1>(vL, vR, eos, F, uf);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) FyH[e * FTX + cc] = F[e];
                    FyH[NEQ * FTX + cc] = uf;
                } else {
                    const int cc = job - 64;
                    const double *pb = P + (HY + TY) * FPX + NG + cc;
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) {
                        const double *s = pb + e * PPL;
                        double unused, v;
                        weno5(s[0], s[-FPX] - s[-2 * FPX], s[0] - s[-FPX], s[FPX] - s[0], s[2 * FPX] - s[FPX], eos.weno_eps4, unused, v);
                        HyR[e * FTX + cc] = v;
                    }
                } }
            }

            // ---- y, first half: reconstruct, publish the right state ----
            double vLy[NEQ];
            if constexpr (D >= 2) {
                double vRy[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double *s = pc + e * PPL;
                    weno5(s[0], s[-FPX] - s[-2 * FPX], s[0] - s[-FPX], s[FPX] - s[0], s[2 * FPX] - s[FPX], eos.weno_eps4, vLy[e], vRy[e]);
                }
#pragma unroll
                for (int e = 0; e < NEQ; ++e) X[e * NT + tid] = vRy[e];
            }
            __syncthreads();                                        // S1: rim results and y right states are visible

            // ---- x: reconstruct, exchange by shuffles, solve face i + 1/2, difference ----
            double acc[NEQ];
            {
                double vL[NEQ], vR[NEQ];
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double *s = pc + e * PPL;
                    weno5(s[0], s[-1] - s[-2], s[0] - s[-1], s[1] - s[0], s[2] - s[1], eos.weno_eps4, vL[e], vR[e]);
                }
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    const double nb = __shfl_down_sync(0xffffffffu, vR[e], 1);
                    vR[e] = i == FTX - 1 ? HxR[e * TY + j] : nb;
                }
                double Fp[NEQ], ufp;
                hllc<D, NF, 0>(vL, vR, eos, Fp, ufp);
                double ufm = __shfl_up_sync(0xffffffffu, ufp, 1);
                if (i == 0) ufm = FxH[NEQ * TY + j];
                const double du = ufp - ufm;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double fm = __shfl_up_sync(0xffffffffu, Fp[e], 1);
                    if (i == 0) fm = FxH[e * TY + j];
                    double rr = fm - Fp[e];
                    if (e >= I::A) rr = fma(pc[e * PPL], du, rr);
                    acc[e] = cx * rr;
                }
            }

            // ---- y, second half: solve face j + 1/2, exchange the flux, difference ----
            if constexpr (D >= 2) {
                double vRn[NEQ], Fy[NEQ], ufy;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) vRn[e] = j == TY - 1 ? HyR[e * FTX + i] : X[e * NT + tid + FTX];
                hllc<D, NF, 1>(vLy, vRn, eos, Fy, ufy);
                __syncthreads();                                    // S2: every right state has been read
#pragma unroll
                for (int e = 0; e < NEQ; ++e) X[e * NT + tid] = Fy[e];
                X[NEQ * NT + tid] = ufy;
                __syncthreads();                                    // S3: fluxes are visible
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

            // ---- a4 + a5: out = ca qn + cb qs + coef (L_x + L_y); the z part follows three planes later ----
            if (active) {
                const long long cell = (D == 3 ? (long long)(p + NG) * g.sz : 0) + col;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double base = 0.0;
                    if (o.nbase > 0) base = o.cb * o.qs[(long long)e * g.cells + cell];
                    if (o.nbase > 1) base = fma(o.ca, o.qn[(long long)e * g.cells + cell], base);
                    o.out[(long long)e * g.cells + cell] = base + acc[e];
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
