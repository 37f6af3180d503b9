// The whole right-hand side L(q) in ONE kernel: ghost fill + cons->prim at load (a0, a1), WENO5 + HLLC in
// x, y and z (a2, a3), flux difference + alpha div u (a4) and the Runge-Kutta stage combine (a5).
//
// Why one kernel.  The path is bound by the FP64 pipe (about 1600 DADD/DMUL/DFMA per cell and evaluation
// against 150 B of compulsory traffic), so every byte that a per-direction design moves
// more than once (primitive array, partial RHS) is time taken from a schedule that has none to spare.  Here a
// cell of q is read once from HBM (plus halo re-reads that hit L2) and a cell of the result is written once.
//
// Decomposition (3D).  A block owns a tile of FTX x TY cells in (x, y) and MARCHES along z over a segment of
// the domain; thread (i, j) = (lane, warp) owns the column (x0 + i, y0 + j).  The z direction runs three
// planes ahead of the in-plane directions, so that when plane ip is differenced in x and y both of its z faces
// are known by the end of the iteration and the cell is written once, complete.  Iteration m, ip = m - 3:
//   * plane ip sits in P with a halo of 3 cells in x and y, laid out by the previous iteration: own cells from
//     the ring of primitive planes (TMEM), halo cells from raw q staged by cp.async two iterations earlier (ghost
//     cells take the wrapped / clamped interior cell);
//   * x: each thread reconstructs its own cell from P; right states and fluxes move between neighbouring
//     lanes by warp shuffles (tile width = warp width);  y: same, through shared memory (right states and fluxes
//     in a buffer each);  the rim of the tile (states of the cells just outside it, in x and in y) is
//     reconstructed by the first four warps, the rim faces are solved by two warps;
//   * while that runs, the raw column of plane m and the raw halo of plane ip + 1 (both landed) are converted
//     to primitives in place (thread-private);
//   * z: cell m - 2 is reconstructed from the thread-private window (planes m - 4, m - 2, m - 1 in the TMEM
//     scratch of the thread, m - 3 in P, m just converted), face (m - 2) - 1/2 solved with the left state parked
//     by the previous iteration and differenced against the previous flux (both in TMEM): the z part of cell ip;
//   * one store: out = ca q_n + cb q_s + coef (L_x + L_y + L_z); q_s staged by cp.async, q_n prefetched into L2;
//   * "glue": P is restaged with plane ip + 1 and the raw reads of the next iterations are issued.  It has no
//     FP64 work, so half of the warps of every scheduler run it before the z part and half after it.
// Every global read is issued at least an iteration before its first use, by the thread that uses it: no block
// barrier is involved in the staging, only cp.async.wait_group.
// FP64 issue needs instruction-level parallelism rather than many warps on this part (one warp per scheduler
// with four independent chains already reaches 92 % of the DFMA peak; weno5 x 7 + hllc alone run at 96 % with
// 8 - 16 warps per SM), so a block is 12 warps with up to 168 registers each.  What the kernel loses
// against that figure is lost where all warps of a scheduler are in non-FP64 code at the same time.
// 1D / 2D: one plane, no march: the same in-plane code on a directly loaded tile.
#pragma once
#include "mfc_math.cuh"

namespace mfc {

#ifndef MFC_XPRE
#define MFC_XPRE 2   // variables whose x reconstruction runs before the first barrier of the in-plane part (measured on the TMA kernel at cfg3: 0: 2.585, 1: 2.563, 2: 2.548, 3: 2.573, 4: 2.572, 6: 2.603, 7: 2.619 ms)
#endif
constexpr int FTX = 32;             // tile width in x = warp width
constexpr int FPX = FTX + 2 * NG;   // staged row length

__device__ __forceinline__ void prefetch_l2(const double *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// ---------------------------------------------------------------------------------------------------------
// shared-memory layout
// ---------------------------------------------------------------------------------------------------------
template <int D, int NF, int TY>
struct FusedCfg {
    static constexpr int NEQ = 2 * NF + D;
    static constexpr int HY = D >= 2 ? NG : 0;
    static constexpr int PY = TY + 2 * HY;
    static constexpr int NT = FTX * TY;
    static constexpr int PPL = PY * FPX;                            // doubles per variable in the staged plane
    static constexpr int NH = PPL - NT;                             // halo cells of the staged plane
    static constexpr int NHT = (NH + NT - 1) / NT;                  // halo cells per thread (at most)
    static constexpr int nP = NEQ * PPL;
    // rim of the tile in x, per row: vL of cell -1, vR of cell 0, vR of cell FTX, flux of lane 0; the rim flux
    // overwrites the first two once they have been read (by the thread that writes it)
    static constexpr int nHx = (3 * NEQ + (NEQ + 1)) * TY;
    // rim in y, per column: vL of row -1, vR of row TY; the rim flux overwrites them likewise
    static constexpr int nHy = D >= 2 ? 2 * NEQ * FTX : 0;
    static constexpr int nX8 = D >= 2 ? NT : 0;                     // face velocity row of the y exchange
    // y exchange: right states X and fluxes X2, [NEQ][NT] each.  X is written before barrier S1 and read between S1 and
    // S2; X2 (and X8) are written before S2 and read after it; both are free again after the barrier that ends the
    // iteration.  3D (cp.async kernel) adds the staging of raw q: own column of the next plane (SQ), q_s of the cell being
    // written (SS), halo cells of the next two staged planes (SH, double buffer).  The z window (ring of four primitive
    // planes, parked left state, previous flux) lives in tensor memory, not here.
    static constexpr int nX = D == 2 ? 2 * NEQ * NT : 0;
    static constexpr int nR = D == 3 ? 2 * NEQ * NT + 2 : 0;        // X, X2 + the TMEM base word
    static constexpr int nS = D == 3 ? NEQ * (2 * NT + 2 * NH) : 0;
    static constexpr int doubles = nP + nHx + nHy + nX8 + nX + nR + nS;
    static constexpr int bytes = doubles * (int)sizeof(double);
    static_assert(TY <= 16, "the x rim jobs are laid out for at most 16 rows");
};

template <int D, int NF, int TY>
struct InplaneBufs {
    const double *P;     // staged plane with halo
    double *X, *X2, *X8; // y exchange: right states [NEQ][NT], fluxes [NEQ][NT] and their face-velocity row [NT]
    double *HxL, *ExR, *HxR, *ExF, *HyL, *HyR;
    __device__ __forceinline__ InplaneBufs(double *P_, double *rim, double *X_, double *X2_, double *X8_) : P(P_), X(X_), X2(X2_), X8(X8_)
    {
        constexpr int NEQ = 2 * NF + D;
        HxL = rim;                    // [NEQ][TY]   left state of face -1/2 (from cell -1)
        ExR = HxL + NEQ * TY;         // [NEQ][TY]   right state of face -1/2 (lane 0)
        HxR = ExR + NEQ * TY;         // [NEQ][TY]   right state of face FTX - 1/2 (from cell FTX)
        ExF = HxR + NEQ * TY;         // [NEQ+1][TY] flux of face 1/2 (lane 0)
        HyL = ExF + (NEQ + 1) * TY;   // [NEQ][FTX]
        HyR = HyL + NEQ * FTX;        // [NEQ][FTX]
    }
};

// ---------------------------------------------------------------------------------------------------------
// a2 + a3 + a4 in x and y on the plane staged in P:  acc[e] += cx L_x + cy L_y  for the thread's cell.
// Called by every thread of the block (it contains two block barriers).
// ---------------------------------------------------------------------------------------------------------
struct NoHook {
    __device__ __forceinline__ void operator()() const {}
};

// non-uniform spacing: coefficient tables of the tile's first own column (x) and row (y), cf. NuRef (mfc_math.cuh)
struct NuPlane {
    const double *tx, *ty;
    int sx, sy;
    __device__ __forceinline__ NuRef x(int col) const { return NuRef{tx + col, sx}; }
    __device__ __forceinline__ NuRef y(int row) const { return NuRef{ty + row, sy}; }
};
// the same for a block that has staged the records (NuRec, mfc_math.cuh) of its columns -1 .. FTX and rows -1 .. TY in
// shared memory: shared-space addresses of the records of column 0 and row 0
struct NuPlaneShared {
    unsigned ax, ay;
    __device__ __forceinline__ NuRec x(int col) const { return NuRec{ax + (unsigned)(col * NU_REC * 8)}; }
    __device__ __forceinline__ NuRec y(int row) const { return NuRec{ay + (unsigned)(row * NU_REC * 8)}; }
};

// `early` runs at the top of the first FP64-heavy block and `mid` at the top of the second: the caller's loads,
// cp.async issues and the cons->prim chains of the NEXT plane go there, so that they overlap this plane's
// arithmetic instead of forming latency-bound phases of their own.
// GT = 0: the two barriers inside are block barriers; GT > 0: barriers of the first GT threads only (bar.sync 1, GT), for
// kernels whose remaining warps run another loop (mfc_fused_roles.cuh)
template <int GT>
__device__ __forceinline__ void inplane_sync()
{
    if constexpr (GT == 0) __syncthreads();
    else asm volatile("bar.sync 1, %0;" ::"n"(GT) : "memory");
}

// ---- rim states.  A unit = ONE variable of one rim cell, one SIDE: (kind, variable e, index r along the rim) with
//   kind 0: left state of y face -1/2 (from row -1)          kind 1: right state of the y face past the tile (row TY)
//   kind 2: left state of x face -1/2 (from cell -1)         kind 3: right state of the x face past the tile (cell FTX)
//   kind 4: right state of x face -1/2 (from cell 0: recomputed here so that the rim face can be solved before lane 0
//           publishes it)
// dealt round-robin to ALL threads (two rounds in 3D with two fluids, the second one leaving out the two warps that
// solve the rim faces), so that no warp reaches the barrier much later than the others.  A right state is the
// left state of the mirrored stencil: one code path, the side only flips the sign of the stride. ----
template <int D, int NF, int TY, int ORDER, bool NU, class NP>
__device__ __forceinline__ void rim_units(const InplaneBufs<D, NF, TY> &B, const Eos &eos, const NP &nup)
{
    using C = FusedCfg<D, NF, TY>;
    constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, HY = C::HY;
    const int tid = threadIdx.x;
    const double *const P = B.P;
    {
        constexpr int UY = D >= 2 ? 2 * FTX * NEQ : 0, UX = 3 * TY * NEQ, U = UY + UX;
#pragma unroll
        for (int u0 = 0; u0 < U; u0 += NT) {
            const int u = u0 + tid;
            if (u < U) {
                int e, r, st;
                const double *pb;
                double *dst;
                decltype(nup.x(0)) nr{};                            // (non-uniform: the rim cell's coefficients)
                if (D >= 2 && u < UY) {
                    const int kind = u / (FTX * NEQ), rem = u - kind * (FTX * NEQ);
                    e = rem / FTX;
                    r = rem - e * FTX;
                    pb = P + e * PPL + (kind == 0 ? HY - 1 : HY + TY) * FPX + NG + r;
                    st = kind == 0 ? FPX : -FPX;
                    dst = (kind == 0 ? B.HyL : B.HyR) + e * FTX + r;
                    if constexpr (NU) nr = nup.y(kind == 0 ? -1 : TY);
                } else {
                    const int v = u - UY, kind = v / (TY * NEQ), rem = v - kind * (TY * NEQ);
                    e = rem / TY;
                    r = rem - e * TY;
                    pb = P + e * PPL + (r + HY) * FPX + NG + (kind == 0 ? -1 : (kind == 1 ? FTX : 0));
                    st = kind == 0 ? 1 : -1;
                    dst = (kind == 0 ? B.HxL : (kind == 1 ? B.HxR : B.ExR)) + e * TY + r;
                    if constexpr (NU) nr = nup.x(kind == 0 ? -1 : (kind == 1 ? FTX : 0));
                }
                double v, other;
                if constexpr (NU) {                                 // the coefficients are not mirror images: both sides, one kept
                    const int sa = st < 0 ? -st : st;
                    reconstruct<ORDER, true>(pb[0], pb[-sa] - pb[-2 * sa], pb[0] - pb[-sa], pb[sa] - pb[0], pb[2 * sa] - pb[sa], eos.weno_eps4, v, other, nr);
                    if (st < 0) v = other;
                } else {
                    reconstruct<ORDER>(pb[0], pb[-st] - pb[-2 * st], pb[0] - pb[-st], pb[st] - pb[0], pb[2 * st] - pb[st], eos.weno_eps4, v, other);
                }
                *dst = v;
            }
        }
    }
}

// the rim faces j = -1/2 (one warp) and i = -1/2 (TY lanes of one warp); the fluxes overwrite the left rim states
template <int D, int NF, int TY>
__device__ __forceinline__ void rim_face_y(const InplaneBufs<D, NF, TY> &B, const Eos &eos)
{
    constexpr int NEQ = 2 * NF + D, NT = FTX * TY;
    const int i = threadIdx.x & 31;
    double *const FyH = B.HyL;
    double hl[NEQ], hr[NEQ], F[NEQ], uf;
#pragma unroll
    for (int e = 0; e < NEQ; ++e) { hl[e] = B.HyL[e * FTX + i]; hr[e] = B.X[e * NT + i]; }
    hllc<D, NF, 1>(hl, hr, eos, F, uf);
#pragma unroll
    for (int e = 0; e < NEQ; ++e) FyH[e * FTX + i] = F[e];
    FyH[NEQ * FTX + i] = uf;
}
template <int D, int NF, int TY>
__device__ __forceinline__ void rim_face_x(const InplaneBufs<D, NF, TY> &B, const Eos &eos)
{
    constexpr int NEQ = 2 * NF + D;
    const int i = threadIdx.x & 31;
    double *const FxH = B.HxL;
    double hl[NEQ], hr[NEQ], F[NEQ], uf;
#pragma unroll
    for (int e = 0; e < NEQ; ++e) { hl[e] = B.HxL[e * TY + i]; hr[e] = B.ExR[e * TY + i]; }
    hllc<D, NF, 0>(hl, hr, eos, F, uf);
#pragma unroll
    for (int e = 0; e < NEQ; ++e) FxH[e * TY + i] = F[e];
    FxH[NEQ * TY + i] = uf;
}

// XP: variables whose x reconstruction runs before barrier S1
template <int D, int NF, int TY, int ORDER, bool NU = false, int GT = 0, int XP = MFC_XPRE, class Early = NoHook, class Mid = NoHook,
          class NP = NuPlane>
__device__ __forceinline__ void inplane_xy(const InplaneBufs<D, NF, TY> &B, const Eos &eos, double cx, double cy,
                                           double (&acc)[2 * NF + D], Early early = Early(), Mid mid = Mid(),
                                           const NP &nup = NP{})
{
    using C = FusedCfg<D, NF, TY>;
    using I = Idx<D, NF>;
    constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, HY = C::HY;
    constexpr int RIMW = TY - 1;                                    // warp that solves the y rim faces
    constexpr int RIMX = TY >= 2 ? TY - 2 : 0;                      // warp that solves the x rim faces
    const int tid = threadIdx.x, i = tid & 31, j = tid >> 5;
    const double *const P = B.P;
    const double *const pc = P + (j + HY) * FPX + (i + NG);         // this thread's cell
    double *const FxH = B.HxL;                                      // [NEQ+1][TY]  flux of face -1/2, over HxL, ExR[0]
    double *const FyH = B.HyL;                                      // [NEQ+1][FTX] over HyL, HyR[0]

    early();
    rim_units<D, NF, TY, ORDER, NU>(B, eos, nup);

    // ---- y, first half: reconstruct, publish the right state ----
    double vLy[NEQ];
    if constexpr (D >= 2) {
        double vRy[NEQ];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            const double *s5 = pc + e * PPL;
            reconstruct<ORDER, NU>(s5[0], s5[-FPX] - s5[-2 * FPX], s5[0] - s5[-FPX], s5[FPX] - s5[0], s5[2 * FPX] - s5[FPX], eos.weno_eps4, vLy[e], vRy[e],
                                   nup.y(j));
        }
#pragma unroll
        for (int e = 0; e < NEQ; ++e) B.X[e * NT + tid] = vRy[e];
    }
    // the x reconstruction needs nothing of the other warps: it runs BEFORE the barrier for the first XPRE variables,
    // so that the barrier's skew and the burst of stencil loads behind it are covered by arithmetic
    constexpr int XPRE = NEQ < XP ? NEQ : XP;
    double vL[NEQ], vR[NEQ];
#pragma unroll
    for (int e = 0; e < XPRE; ++e) {
        const double *s5 = pc + e * PPL;
        reconstruct<ORDER, NU>(s5[0], s5[-1] - s5[-2], s5[0] - s5[-1], s5[1] - s5[0], s5[2] - s5[1], eos.weno_eps4, vL[e], vR[e], nup.x(i));
    }
    inplane_sync<GT>();                                             // S1: rim states and y right states are visible

    // ---- x: reconstruct, exchange by shuffles, solve face i + 1/2, difference ----
    mid();
    double ax[NEQ];
    {
#pragma unroll
        for (int e = XPRE; e < NEQ; ++e) {
            const double *s5 = pc + e * PPL;
            reconstruct<ORDER, NU>(s5[0], s5[-1] - s5[-2], s5[0] - s5[-1], s5[1] - s5[0], s5[2] - s5[1], eos.weno_eps4, vL[e], vR[e], nup.x(i));
        }
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            const double nb = __shfl_down_sync(0xffffffffu, vR[e], 1);
            vR[e] = i == FTX - 1 ? B.HxR[e * TY + j] : nb;
        }
        double Fp[NEQ], ufp;
        hllc<D, NF, 0>(vL, vR, eos, Fp, ufp);
        if (i == 0) {
#pragma unroll
            for (int e = 0; e < NEQ; ++e) B.ExF[e * TY + j] = Fp[e];
            B.ExF[NEQ * TY + j] = ufp;
        }
        const double du = ufp - __shfl_up_sync(0xffffffffu, ufp, 1);
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            double rr = __shfl_up_sync(0xffffffffu, Fp[e], 1) - Fp[e];
            if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, pc[e * PPL], pc[I::E * PPL]), du, rr);
            ax[e] = rr;                                             // lane 0 is redone below with the rim flux
        }
    }

    // ---- y, second half: solve face j + 1/2 (and, one warp, the rim faces j = -1/2) ----
    double Fy[NEQ], ufy = 0.0;
    if constexpr (D >= 2) {
        double vRn[NEQ];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) vRn[e] = j == TY - 1 ? B.HyR[e * FTX + i] : B.X[e * NT + tid + FTX];
        hllc<D, NF, 1>(vLy, vRn, eos, Fy, ufy);
        if (j == RIMW) rim_face_y<D, NF, TY>(B, eos);
    }
    if (j == RIMX && i < TY) rim_face_x<D, NF, TY>(B, eos);                 // rim faces i = -1/2, one per row
    if constexpr (D >= 2) {                                         // the fluxes have a buffer of their own: no barrier before this
#pragma unroll
        for (int e = 0; e < NEQ; ++e) B.X2[e * NT + tid] = Fy[e];
        B.X8[tid] = ufy;
    }
    inplane_sync<GT>();                                             // S2: fluxes (rim ones included) are visible
    if (i == 0) {
        const double du = B.ExF[NEQ * TY + j] - FxH[NEQ * TY + j];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            double rr = FxH[e * TY + j] - B.ExF[e * TY + j];
            if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, pc[e * PPL], pc[I::E * PPL]), du, rr);
            ax[e] = rr;
        }
    }
#pragma unroll
    for (int e = 0; e < NEQ; ++e) acc[e] = fma(cx, ax[e], acc[e]);
    if constexpr (D >= 2) {
        const double ufm = j == 0 ? FyH[NEQ * FTX + i] : B.X8[tid - FTX];
        const double du = ufy - ufm;
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            const double fm = j == 0 ? FyH[e * FTX + i] : B.X2[e * NT + tid - FTX];
            double rr = fm - Fy[e];
            if (e >= I::A) rr = fma(alpha_div_coef<NF>(eos, pc[e * PPL], pc[I::E * PPL]), du, rr);
            acc[e] = fma(cy, rr, acc[e]);
        }
    }
}

// source cell of staged position (ii, jj) of plane p: ghost fill = index map
template <int D>
__device__ __forceinline__ long long staged_source(const Geo &g, int x0, int y0, int p, int ii, int jj)
{
    long long src = bc_source(min(x0 - NG + ii, g.n[0] + NG - 1), g.n[0], g.bc_lo[0], g.bc_hi[0]) + NG;
    if (D >= 2) src += (long long)(bc_source(min(y0 - NG + jj, g.n[1] + NG - 1), g.n[1], g.bc_lo[1], g.bc_hi[1]) + NG) * g.sy;
    if (D == 3) src += (long long)(bc_source(min(max(p, -NG), g.n[2] + NG - 1), g.n[2], g.bc_lo[2], g.bc_hi[2]) + NG) * g.sz;
    return src;
}

// ---------------------------------------------------------------------------------------------------------
// 1D and 2D: one tile per block
// ---------------------------------------------------------------------------------------------------------
template <int D, int NF, int TY, int ORDER, bool NU>
__global__ void __launch_bounds__(FTX *TY, 1)
    rhs_fused_plane_kernel(typename GeoOf<NU>::type g, Eos eos, const double *__restrict__ q, SweepOut o, int ntx)
{
    static_assert(D <= 2, "plane kernel");
    using C = FusedCfg<D, NF, TY>;
    constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL;
    extern __shared__ double sm[];
    double *const P = sm;
    double *const rim = P + C::nP;
    double *const X8 = rim + C::nHx + C::nHy;
    double *const X = X8 + C::nX8;
    const InplaneBufs<D, NF, TY> B(P, rim, X, X + NEQ * NT, X8);

    const int tid = threadIdx.x, i = tid & 31, j = tid >> 5;
    const int bx = blockIdx.x % ntx, by = blockIdx.x / ntx;
    const int x0 = bx * FTX, y0 = by * TY;
    const bool active = x0 + i < g.n[0] && (D < 2 || y0 + j < g.n[1]);
    const long long cell = (long long)(x0 + i + NG) + (D >= 2 ? (long long)(y0 + j + NG) * g.sy : 0);

    for (int c = tid; c < PPL; c += NT) {
        const int jj = c / FPX, ii = c - jj * FPX;
        const long long src = staged_source<D>(g, x0, y0, 0, ii, jj);
        double qc[NEQ], wc[NEQ];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) qc[e] = __ldg(q + (long long)e * g.cells + src);
        cons_to_prim_cell<D, NF>(qc, eos, wc);
#pragma unroll
        for (int e = 0; e < NEQ; ++e) P[e * PPL + c] = wc[e];
    }
    __syncthreads();
    double acc[NEQ];
#pragma unroll
    for (int e = 0; e < NEQ; ++e) acc[e] = 0.0;
    if constexpr (NU) {   // per-cell widths and coefficient tables (rows of stride g.nus[d], padded past the last cell)
        const NuPlane nup{g.nu[0] + x0 + NG, D >= 2 ? g.nu[1] + y0 + NG : nullptr, g.nus[0], g.nus[1]};
        inplane_xy<D, NF, TY, ORDER, true>(B, eos, o.coef * __ldg(nup.tx + i + 27 * nup.sx), D >= 2 ? o.coef * __ldg(nup.ty + j + 27 * nup.sy) : 0.0, acc,
                                           NoHook(), NoHook(), nup);
    } else {
        inplane_xy<D, NF, TY, ORDER>(B, eos, o.coef * g.inv_dx[0], D >= 2 ? o.coef * g.inv_dx[1] : 0.0, acc);
    }
    if (active) {
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            double v = acc[e];
            if (o.nbase > 0) v = fma(o.cb, o.qs[(long long)e * g.cells + cell], v);
            if (o.nbase > 1) v = fma(o.ca, o.qn[(long long)e * g.cells + cell], v);
            o.out[(long long)e * g.cells + cell] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Tensor memory (TMEM, 256 KB per SM) as thread-private scratch.  Nothing on this path uses the tensor cores, so
// the whole of it is free: the z window of a column (ring of primitive planes), the parked left state, the
// previous z flux and the plane that left the ring live there instead of in shared memory and registers.
// A warp reaches the 32 TMEM lanes of its quarter (warp index mod 4), one lane per thread; the warps of a quarter
// take disjoint column ranges.  tcgen05.ld / st with shape 32x32b move N consecutive 32-bit columns of the
// thread's own lane to / from registers.  TV = values (doubles) per slot: 8 (x16) or 10 (x16 + x4, three fluids).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc512(unsigned *smem_word)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((unsigned)__cvta_generic_to_shared(smem_word)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc512(unsigned base)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base) : "memory");
}
template <int TV>
__device__ __forceinline__ void tmem_load(unsigned a, double (&v)[TV])
{
    static_assert(TV == 8 || TV == 10, "8 doubles (x16) or 10 doubles (x16 + x4) per transfer");
    unsigned r[2 * TV];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(a));
    if constexpr (TV == 10) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]) : "r"(a + 16u));
    }
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int k = 0; k < TV; ++k) v[k] = __hiloint2double((int)r[2 * k + 1], (int)r[2 * k]);
}
template <int TV>
__device__ __forceinline__ void tmem_store(unsigned a, const double (&v)[TV])
{
    unsigned r[2 * TV];
#pragma unroll
    for (int k = 0; k < TV; ++k) { r[2 * k] = (unsigned)__double2loint(v[k]); r[2 * k + 1] = (unsigned)__double2hiint(v[k]); }
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(a), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
                   "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
                 : "memory");
    if constexpr (TV == 10) {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"
                     ::"r"(a + 16u), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]) : "memory");
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// ---------------------------------------------------------------------------------------------------------
// 3D: tile in (x, y), march along z
// ---------------------------------------------------------------------------------------------------------
template <int NF, int TY, int ORDER, bool NU>
__global__ void __launch_bounds__(FTX *TY, 1)
    rhs_fused_march_kernel(typename GeoOf<NU>::type g, Eos eos, const double *__restrict__ q, SweepOut o, int ntx, int nty, int seg)
{
    constexpr int D = 3;
    using C = FusedCfg<D, NF, TY>;
    using I = Idx<D, NF>;
    constexpr int NEQ = C::NEQ, NT = C::NT, PPL = C::PPL, NH = C::NH, NHT = C::NHT;
    extern __shared__ double sm[];
    double *const P = sm;
    double *const rim = P + C::nP;
    double *const X8 = rim + C::nHx + C::nHy;
    double *const X = X8 + C::nX8;                                  // [NEQ][NT]    y exchange
    double *const X2 = X + NEQ * NT;                                // [NEQ][NT]    y exchange, fluxes
    double *const SQ = X2 + NEQ * NT;                               // [NEQ][NT]    raw q, own column, next plane
    double *const SS = SQ + NEQ * NT;                               // [NEQ][NT]    raw q_s of the cell being written
    double *const SH = SS + NEQ * NT;                               // [2][NEQ][NH] raw q, halo cells of the next two staged planes
    unsigned *const tmem_word = reinterpret_cast<unsigned *>(SH + 2 * NEQ * NH);
    // thread-private TMEM scratch (see above): slots of TV doubles = 2 TV columns each
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
    // own column as a SOURCE (a thread past the domain edge still computes on admissible data)
    const int scol = (int)staged_source<2>(g, x0, y0, 0, i + NG, j + NG);   // == the own cell for an active thread
    const int col = scol;
    double *const pcw = P + (j + NG) * FPX + (i + NG);
    // halo cells of this thread: staged position.  Halo positions are numbered in row-major order of the staged
    // plane, skipping the interior block.
    int hpos[NHT];
#pragma unroll
    for (int t = 0; t < NHT; ++t) {
        const int h = tid + t * NT;
        constexpr int TOP = NG * FPX;                               // cells of the full rows above (below) the tile
        int c = 0;
        if (h < TOP) c = h;
        else if (h < TOP + 2 * NG * TY) {
            const int r = (h - TOP) / (2 * NG), k = (h - TOP) - r * 2 * NG;
            c = (NG + r) * FPX + (k < NG ? k : FTX + k);
        } else if (h < NH) c = (NG + TY) * FPX + (h - TOP - 2 * NG * TY);
        hpos[t] = c;
    }
    auto zoff = [&](int p) -> long long {
        return (long long)(bc_source(min(max(p, -NG), g.n[2] + NG - 1), g.n[2], g.bc_lo[2], g.bc_hi[2]) + NG) * g.sz;
    };
    auto stage_column = [&](int p) {                                // raw q of plane p, own column -> SQ
        const double *src = q + zoff(p) + scol;
#pragma unroll
        for (int e = 0; e < NEQ; ++e) cp_async8(SQ + e * NT + tid, src + (long long)e * g.cells);
    };
    auto stage_halo = [&](int p) {                                  // raw q of plane p, this thread's halo cells -> SH[p & 1]
        const long long zo = zoff(p);
        double *const sh = SH + (p & 1) * NEQ * NH;
#pragma unroll
        for (int t = 0; t < NHT; ++t) {
            if (tid + t * NT < NH) {
                const int jj = hpos[t] / FPX, ii = hpos[t] - jj * FPX;
                const double *src = q + zo + staged_source<2>(g, x0, y0, 0, ii, jj);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) cp_async8(sh + e * NH + t * NT + tid, src + (long long)e * g.cells);
            }
        }
    };
    auto stage_base = [&](int p) {                                  // raw q_s of cell (own column, plane p) -> SS
        if (o.nbase > 0 && active) {
            const double *src = o.qs + (long long)(p + NG) * g.sz + col;
#pragma unroll
            for (int e = 0; e < NEQ; ++e) cp_async8(SS + e * NT + tid, src + (long long)e * g.cells);
        }
    };

    // TMEM: one warp allocates all 512 columns (one block per SM), everybody reads the base after a barrier
    if (j == 0) tmem_alloc512(tmem_word);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem_base = *tmem_word;
    // this thread's scratch: lane = 32 (warp mod 4) + lane id (implied by the 32x32b shape), columns by warp / 4
    const unsigned tbase = tmem_base + ((unsigned)(32 * (j & 3)) << 16) + (unsigned)((j >> 2) * T_SLOTS * 2 * TV);
    auto tslot = [&](int s) -> unsigned { return tbase + (unsigned)(s * 2 * TV); };
    {   // previous z flux (T_FLUX: NEQ fluxes + the face velocity) and the plane that left the ring (T_PREV) start at zero
        double z[TV];
#pragma unroll
        for (int k = 0; k < TV; ++k) z[k] = 0.0;
        tmem_store<TV>(tslot(T_FLUX), z);
        tmem_store<TV>(tslot(T_PREV), z);
    }

    // cons->prim of the staged raw values, in place and thread-private: own column of the next plane (SQ) and this
    // thread's halo cells of the next staged plane (SH)
    auto convert_staged = [&](bool column, int hplane) {            // hplane < 0: no halo to convert
        if (column) {
            double qc[NEQ], wc[NEQ];
#pragma unroll
            for (int e = 0; e < NEQ; ++e) qc[e] = SQ[e * NT + tid];
            cons_to_prim_cell<D, NF>(qc, eos, wc);
#pragma unroll
            for (int e = 0; e < NEQ; ++e) SQ[e * NT + tid] = wc[e];
        }
        if (hplane >= 0) {
            double *const sh = SH + (hplane & 1) * NEQ * NH;
#pragma unroll
            for (int t = 0; t < NHT; ++t) {
                if (tid + t * NT < NH) {
                    double qc[NEQ], wc[NEQ];
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) qc[e] = sh[e * NH + t * NT + tid];
                    cons_to_prim_cell<D, NF>(qc, eos, wc);
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) sh[e * NH + t * NT + tid] = wc[e];
                }
            }
        }
    };

    // Iteration m: plane ip = m - 3 (staged in P by the previous iteration) is differenced in x and y; then plane m
    // enters the z window, cell m - 2 is reconstructed, face (m - 2) - 1/2 solved, and cell ip is complete.
    //   in-plane (three barriers): q_n of the next plane prefetched at its top; in its second block the raw column m
    //            (SQ) and the raw halo of plane ip + 1 (SH) are converted to primitives in place
    //   bottom   z part from wn = SQ; plane m -> ring; out(ip) written  ||  glue: P restaged with plane ip + 1 (own
    //            cell from the ring, halo cells from SH); issue, as three commit groups in this order, {q_s of cell
    //            ip + 1}, {raw column m + 1}, {raw halo of plane m = ip + 3}   (order of the two halves per warp group)
    //   barrier  (P is staged; X, X2 and the rim buffers are free again)
    // The conversions need everything but the youngest group (the halo issued one iteration ago is used two
    // iterations after its issue), so the only wait is "all but the youngest", half an iteration after the issue
    // of q_s (L2-resident: it was this block's column three planes ago) and of the column.
    const int pstart = k0 - NG, pend = k1 + NG;
    cp_async_commit();
    stage_column(pstart);
    cp_async_commit();
    cp_async_commit();
#pragma unroll 1
    for (int m = pstart; m < pend; ++m) {
        const int n = m - pstart;                                   // planes brought in before this one
        const int ip = m - NG;
        const bool inplane = ip >= k0;                              // block-uniform (ip < k1 always)
        const bool next_inplane = ip + 1 >= k0 && ip + 1 < k1;
        const long long cell = (long long)(ip + NG) * g.sz + col;
        // the three coefficients are re-read from the constant bank every iteration rather than held in registers
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

        double acc[NEQ];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) acc[e] = 0.0;
        if (inplane) {
            auto early = [&]() {                                    // q_n of the next plane: into L2
                if (active && o.nbase > 1 && ip + 1 < k1) {
#pragma unroll
                    for (int e = 0; e < NEQ; ++e) prefetch_l2(o.qn + (long long)e * g.cells + cell + g.sz);
                }
            };
            auto mid = [&]() {                                      // q_s, column m and the halo of plane ip + 1 have landed
                cp_async_wait<1>();
                convert_staged(true, next_inplane ? ip + 1 : -1);
            };
            const InplaneBufs<D, NF, TY> B(P, rim, X, X2, X8);
            inplane_xy<D, NF, TY, ORDER, NU>(B, eos, cx, cy, acc, early, mid, nup);
        } else {
            cp_async_wait<1>();
            convert_staged(true, next_inplane ? ip + 1 : -1);
        }

        // ---- bottom of the iteration.  q_n (in L2 since the previous iteration) is loaded now and used at the very
        // end; q_s joins the in-plane part at once ----
        double qnv[NEQ];
        if (inplane && active) {
            if (o.nbase > 1) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e) qnv[e] = __ldcg(o.qn + (long long)e * g.cells + cell);
            }
            if (o.nbase > 0) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e) acc[e] = fma(o.cb, SS[e * NT + tid], acc[e]);
            }
        }
        // plane m of the own column (primitives since the conversion above) and plane m - 3 = ip: the latter sits in P
        // when it has just been differenced in plane, else in its ring slot
        double wn[TV], vb[TV];
#pragma unroll
        for (int k = NEQ; k < TV; ++k) { wn[k] = 0.0; vb[k] = 0.0; }
#pragma unroll
        for (int e = 0; e < NEQ; ++e) wn[e] = SQ[e * NT + tid];
        if (inplane) {
#pragma unroll
            for (int e = 0; e < NEQ; ++e) vb[e] = pcw[e * PPL];
        } else if (n >= 3) {
            tmem_load<TV>(tslot(T_RING + ((m + 1) & 3)), vb);
        } else {
#pragma unroll
            for (int e = 0; e < NEQ; ++e) vb[e] = 0.0;
        }
        // "glue": plane ip + 1 -> P, raw reads of the next iterations issued.  No FP64 work: half of the warps of every
        // scheduler run it BEFORE the z part and half AFTER it, so that it overlaps the other half's arithmetic
        auto glue = [&]() {
            if (next_inplane) {
                double rp[TV];                                      // plane m - 2 = ip + 1
                tmem_load<TV>(tslot(T_RING + ((m + 2) & 3)), rp);
#pragma unroll
                for (int e = 0; e < NEQ; ++e) pcw[e * PPL] = rp[e];
                const double *const sh = SH + ((ip + 1) & 1) * NEQ * NH;
#pragma unroll
                for (int t = 0; t < NHT; ++t) {
                    if (tid + t * NT < NH) {
#pragma unroll
                        for (int e = 0; e < NEQ; ++e) P[e * PPL + hpos[t]] = sh[e * NH + t * NT + tid];
                    }
                }
                stage_base(ip + 1);
            }
            cp_async_commit();
            if (m + 1 < pend) stage_column(m + 1);
            cp_async_commit();
            if (m >= k0 && m < k1) stage_halo(m);                   // plane ip + 3: the buffer the copy above just freed
            cp_async_commit();
            if (m + 2 < pend) {                                     // the column after that: into L2
                const double *src = q + zoff(m + 2) + scol;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) prefetch_l2(src + (long long)e * g.cells);
            }
        };
        auto zpart = [&]() {
            // ---- z: reconstruct cell m - 2, solve face (m - 2) - 1/2, difference for cell m - 3 = ip ----
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
                    double Fm[TV], Fn[TV];                          // previous and new flux; entry NEQ is the face velocity
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
                        acc[e] = fma(cz, rr, acc[e]);               // meaningful when c > k0, i.e. when ip >= k0
                        Fn[e] = Fp[e];
                    }
                    Fn[NEQ] = ufp;
                    tmem_store<TV>(tslot(T_FLUX), Fn);
                }
            }
            tmem_store<TV>(tslot(T_PREV), vb);
            // plane m enters the ring: the slot of plane m - 4
            tmem_store<TV>(tslot(T_RING + (m & 3)), wn);
            // ---- a5: out = ca q_n + cb q_s + coef L ----
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
        __syncthreads();                                            // P is staged; X, X2 and the rim buffers are free
    }
    if (j == 0) tmem_dealloc512(tmem_base);
}

}  // namespace mfc
