// Kernels of the hot path: cons->prim with ghost fill, the fused WENO5 + HLLC + flux-difference sweeps in x
// (tile + neighbour exchange) and y / z (marching), the CFL reduction, and the one-line stage kernels.
// Sweeps stage their stencil data in shared memory with cp.async so that loads in flight hold no registers.
#pragma once
#include "mfc_math.cuh"

namespace mfc {

// a0 + a1: one thread per padded cell; ghost cells read the wrapped / clamped interior cell
template <int D, int NF>
__global__ void __launch_bounds__(256) prim_kernel(Geo g, Eos eos, const double *__restrict__ q, double *__restrict__ w)
{
    using I = Idx<D, NF>;
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= g.cells) return;
    const int i = (int)(c % g.p[0]);
    const long long r = c / g.p[0];
    const int j = (int)(r % g.p[1]);
    const int k = (int)(r / g.p[1]);
    const int si = bc_source(i - g.g[0], g.n[0], g.bc_lo[0], g.bc_hi[0]) + g.g[0];
    const int sj = D > 1 ? bc_source(j - g.g[1], g.n[1], g.bc_lo[1], g.bc_hi[1]) + g.g[1] : 0;
    const int sk = D > 2 ? bc_source(k - g.g[2], g.n[2], g.bc_lo[2], g.bc_hi[2]) + g.g[2] : 0;
    const long long src = (long long)sk * g.sz + (long long)sj * g.sy + si;
    double qc[I::NEQ], wc[I::NEQ];
#pragma unroll
    for (int e = 0; e < I::NEQ; ++e) qc[e] = __ldg(q + (long long)e * g.cells + src);
    cons_to_prim_cell<D, NF>(qc, eos, wc);
#pragma unroll
    for (int e = 0; e < I::NEQ; ++e) w[(long long)e * g.cells + c] = wc[e];
}

// ---------------------------------------------------------------------------------------------------------
// x sweep (first sweep of every L evaluation).  Persistent blocks walk over tiles of the STAGED index space
//   g = row * px + ipad,   row = interior (y, z) line, ipad = padded x index,
// which is contiguous in memory inside a z plane, so a tile of XT + 4 staged values per primitive is one
// contiguous run (ghost cells of the primitive array are already filled).  Thread t owns staged position
// g0 + 2 + t: it reads its 5-cell stencil from shared memory, reconstructs both face states, takes the right
// state of face t+1/2 from thread t+1 and the flux of face t-1/2 from thread t-1 through shared memory, and
// writes its own cell.  Threads 0 and XT-1 only feed their neighbours, so tiles advance by XT - 2.
// The next tile's values are copied with cp.async while the current tile is computed (double buffer); the
// per-cell streams of the output stage (qs, qn) are copied the same way at the top of the tile's iteration
// and consumed at its end.
// ---------------------------------------------------------------------------------------------------------
constexpr int XT = 256;          // threads per block = reconstructed cells per tile
constexpr int XS = XT + 4;       // staged values per primitive per tile

template <int NEQ>
constexpr int sweep_x_smem_bytes() { return (2 * NEQ * XS + 2 * NEQ * XT + NEQ * XT + (NEQ + 1) * XT) * (int)sizeof(double); }

template <int D, int NF>
__global__ void __launch_bounds__(XT, 2) sweep_x_kernel(Geo g, Eos eos, const double *__restrict__ w, SweepOut o, int ntiles)
{
    using I = Idx<D, NF>;
    constexpr int NEQ = I::NEQ;
    extern __shared__ double smem[];
    double *stage = smem;                       // [2][NEQ][XS]
    double *aux = stage + 2 * NEQ * XS;         // [2][NEQ][XT] : qs, qn of the thread's own cell
    double *exR = aux + 2 * NEQ * XT;           // [NEQ][XT]    : right states
    double *exF = exR + NEQ * XT;               // [NEQ + 1][XT]: fluxes and face velocity
    const int t = threadIdx.x;
    const int px = g.p[0], ny = g.n[1];
    const long long G = (long long)g.n[1] * g.n[2] * px;
    const double c1 = o.coef * g.inv_dx[0];

    // copies the staged values [g0, g0 + XS) of every primitive into buffer `buf`
    auto issue_stage = [&](int tile, int buf) {
        const long long g0 = (long long)tile * (XT - 2);
        for (int s = t; s < XS; s += XT) {
            const long long gg = g0 + s;
            if (gg < G) {
                const long long row = gg / px;
                const int ip = (int)(gg - row * px);
                const int j = (int)(row % ny), kk = (int)(row / ny);
                const double *src = w + (long long)(kk + g.g[2]) * g.sz + (long long)(j + g.g[1]) * g.sy + ip;
                double *dst = stage + buf * NEQ * XS + s;
#pragma unroll
                for (int e = 0; e < NEQ; ++e) cp_async8(dst + e * XS, src + (long long)e * g.cells);
            }
        }
    };

    int tile = blockIdx.x, buf = 0;
    if (tile < ntiles) issue_stage(tile, 0);
    cp_async_commit();
    for (; tile < ntiles; tile += gridDim.x, buf ^= 1) {
        // this thread's cell
        const long long gt = (long long)tile * (XT - 2) + 2 + t;
        const long long row = gt / px;
        const int ip = (int)(gt - row * px);
        const int j = (int)(row % ny), kk = (int)(row / ny);
        const long long cell = (long long)(kk + g.g[2]) * g.sz + (long long)(j + g.g[1]) * g.sy + ip;
        const bool emit = gt < G && ip >= NG && ip <= px - NG - 1 && t >= 1 && t <= XT - 2;
        if (emit && o.nbase > 0) {
#pragma unroll
            for (int e = 0; e < NEQ; ++e) cp_async8(aux + e * XT + t, o.qs + (long long)e * g.cells + cell);
            if (o.nbase > 1) {
#pragma unroll
                for (int e = 0; e < NEQ; ++e) cp_async8(aux + (NEQ + e) * XT + t, o.qn + (long long)e * g.cells + cell);
            }
        }
        cp_async_commit();
        const int next = tile + gridDim.x;
        if (next < ntiles) issue_stage(next, buf ^ 1);
        cp_async_commit();
        cp_async_wait<2>();                      // this tile's staged values (committed one iteration ago) have landed
        __syncthreads();

        const double *st = stage + buf * NEQ * XS + t;
        double vL[NEQ], vR[NEQ], acell[I::NA > 0 ? I::NA : 1];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            const double *p = st + e * XS;
            const double a = p[0], b = p[1], c = p[2], d = p[3], ee = p[4];
            weno5(c, b - a, c - b, d - c, ee - d, eos.weno_eps4, vL[e], vR[e]);
            if (e >= I::A) acell[e - I::A] = c;
            exR[e * XT + t] = vR[e];
        }
        __syncthreads();
        const int tn = t + 1 < XT ? t + 1 : t;
#pragma unroll
        for (int e = 0; e < NEQ; ++e) vR[e] = exR[e * XT + tn];
        double Fp[NEQ], ufp;
        hllc<D, NF, 0>(vL, vR, eos, Fp, ufp);       // face t + 1/2
#pragma unroll
        for (int e = 0; e < NEQ; ++e) exF[e * XT + t] = Fp[e];
        exF[NEQ * XT + t] = ufp;
        cp_async_wait<1>();                      // qs, qn of this tile
        __syncthreads();
        if (emit) {
            const double du = ufp - exF[NEQ * XT + t - 1];
#pragma unroll
            for (int e = 0; e < NEQ; ++e) {
                double r = exF[e * XT + t - 1] - Fp[e];
                if (e >= I::A) r = fma(acell[e - I::A], du, r);
                double base = 0.0;
                if (o.nbase > 0) base = o.cb * aux[e * XT + t];
                if (o.nbase > 1) base = fma(o.ca, aux[(NEQ + e) * XT + t], base);
                o.out[(long long)e * g.cells + cell] = fma(c1, r, base);
            }
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------------------
// y / z sweep without transposes: threads span the flattened (x, other transverse index, segment) space so
// that a warp reads 32 consecutive x (coalesced), and each thread MARCHES along the sweep direction.  The
// 5-plane stencil window of every primitive lives in a per-thread ring in shared memory that cp.async fills
// MA planes ahead of use: loads in flight hold no registers and a thread never waits on a load it has just
// issued.  A thread only ever reads its own column of the ring, so the kernel has no block-level barrier.
// The left state of the previous face is handed from one iteration to the next through shared memory and
// the previous flux through registers, so each cell of a segment is read once and reconstructed once; a
// segment of S cells costs S + 2 reconstructions and S + 1 Riemann problems.
// out[cell] += coef * L_dir (SweepOut, first == 0).
// ---------------------------------------------------------------------------------------------------------
constexpr int MBT = 128;         // threads per block
constexpr int MA = 1;            // planes in flight beyond the stencil window
constexpr int MR = 5 + MA;       // ring slots

template <int NEQ>
constexpr int sweep_march_smem_bytes() { return (MR + 2) * NEQ * MBT * (int)sizeof(double); }

template <int D, int NF, int DIR>
__global__ void __launch_bounds__(MBT, 4) sweep_march_kernel(Geo g, Eos eos, const double *__restrict__ w, SweepOut o,
                                                             int seg, int nseg)
{
    using I = Idx<D, NF>;
    constexpr int NEQ = I::NEQ;
    static_assert(DIR == 1 || DIR == 2, "marching sweeps are y and z");
    constexpr int OTH = DIR == 1 ? 2 : 1;                 // the other transverse dimension
    constexpr int SLOT = NEQ * MBT;                       // doubles per ring slot
    extern __shared__ double smem[];
    double *ring = smem + threadIdx.x;                    // [MR][NEQ][MBT], this thread's column
    double *park = ring + MR * SLOT;                      // [NEQ][MBT]: left state of the previous face
    double *obuf = park + SLOT;                           // [NEQ][MBT]: out values of the cell about to be updated
    const int nx = g.n[0], no = g.n[OTH], nm = g.n[DIR];
    const long long gidx = (long long)blockIdx.x * MBT + threadIdx.x;
    if (gidx >= (long long)nx * no * nseg) return;        // no block-level barrier below
    const int i = (int)(gidx % nx);
    const long long r = gidx / nx;
    const int oo = (int)(r % no);
    const int s = (int)(r / no);
    const int j0 = s * seg;
    const int j1 = min(j0 + seg, nm);
    const long long sm = DIR == 1 ? g.sy : g.sz;          // stride along the march
    const long long so = DIR == 1 ? g.sz : g.sy;
    // plane n (n = 0 .. np-1) of this thread is the cell with march index j0 - 3 + n; centre cells run j0-1 .. j1
    const int np = j1 - j0 + 6;
    const long long col = (long long)(i + NG) + (long long)(oo + g.g[OTH]) * so;
    const double *src = w + col + (long long)(j0 - 3 + NG) * sm;      // next plane to copy
    double *outp = o.out + col + (long long)(j0 - 1 + NG) * sm;       // cell of the current centre
    const double c1 = o.coef * g.inv_dx[DIR];

    int nissued = 0, wslot = 0;                           // planes issued; ring slot the next plane goes to
    auto issue_plane = [&]() {
        if (nissued < np) {
            double *dst = ring + wslot * SLOT;
#pragma unroll
            for (int e = 0; e < NEQ; ++e) cp_async8(dst + e * MBT, src + (long long)e * g.cells);
            src += sm;
        }
        ++nissued;
        wslot = wslot + 1 == MR ? 0 : wslot + 1;
        cp_async_commit();
    };
#pragma unroll 1
    for (int n = 0; n < MR - 1; ++n) issue_plane();

    double Fm[NEQ], ufm = 0.0;
#pragma unroll
    for (int e = 0; e < NEQ; ++e) Fm[e] = 0.0;
    int s0 = 0;                                           // ring slot of the oldest plane of the window
#pragma unroll 1
    for (int k = j0 - 1; k <= j1; ++k, outp += sm) {
        if (k > j0) {                                     // out values of cell k - 1, consumed at the end of this iteration
            const double *ob = outp - sm;
#pragma unroll
            for (int e = 0; e < NEQ; ++e) cp_async8(obuf + e * MBT, ob + (long long)e * g.cells);
        }
        issue_plane();                                    // into the slot the previous iteration's oldest plane left
        cp_async_wait<MA>();                              // planes k-2 .. k+2 have landed
        int sl[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) { const int v = s0 + q; sl[q] = (v >= MR ? v - MR : v) * SLOT; }
        s0 = s0 + 1 == MR ? 0 : s0 + 1;

        double vLp[NEQ], vR[NEQ];
#pragma unroll
        for (int e = 0; e < NEQ; ++e) {
            const double a = ring[sl[0] + e * MBT], b = ring[sl[1] + e * MBT], c = ring[sl[2] + e * MBT];
            const double d = ring[sl[3] + e * MBT], ee = ring[sl[4] + e * MBT];
            double vL;
            weno5(c, b - a, c - b, d - c, ee - d, eos.weno_eps4, vL, vR[e]);
            vLp[e] = park[e * MBT];                       // left state of face k - 1/2 (from cell k - 1)
            park[e * MBT] = vL;                           // left state of face k + 1/2, for the next iteration
        }
        if (k >= j0) {
            double Fp[NEQ], ufp;
            hllc<D, NF, DIR>(vLp, vR, eos, Fp, ufp);      // face k - 1/2
            if (k > j0) {                                 // cell k - 1: its centre plane is the window's second slot
                double *op = outp - sm;
                const double du = ufp - ufm;
                cp_async_wait<0>();                       // obuf has landed
#pragma unroll
                for (int e = 0; e < NEQ; ++e) {
                    double rr = Fm[e] - Fp[e];
                    if (e >= I::A) rr = fma(ring[sl[1] + e * MBT], du, rr);
                    op[(long long)e * g.cells] = fma(c1, rr, obuf[e * MBT]);
                }
            }
#pragma unroll
            for (int e = 0; e < NEQ; ++e) Fm[e] = Fp[e];
            ufm = ufp;
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------------------
// a6 CFL: min over interior cells and directions of dx_d / (|u_d| + c).  Positive doubles
// order like their bit patterns, so the grid-wide minimum is an integer atomicMin.
// ---------------------------------------------------------------------------------------------------------
template <int D, int NF>
__global__ void __launch_bounds__(256) cfl_kernel(Geo g, Eos eos, const double *__restrict__ q, unsigned long long *min_bits)
{
    using I = Idx<D, NF>;
    const long long ncell = (long long)g.n[0] * g.n[1] * g.n[2];
    double best = 1.0e300;
    for (long long f = (long long)blockIdx.x * blockDim.x + threadIdx.x; f < ncell; f += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(f % g.n[0]);
        const long long r = f / g.n[0];
        const int j = (int)(r % g.n[1]), k = (int)(r / g.n[1]);
        const long long cell = (long long)(k + g.g[2]) * g.sz + (long long)(j + g.g[1]) * g.sy + (i + NG);
        double qc[I::NEQ], wc[I::NEQ];
#pragma unroll
        for (int e = 0; e < I::NEQ; ++e) qc[e] = __ldg(q + (long long)e * g.cells + cell);
        cons_to_prim_cell<D, NF>(qc, eos, wc);
        double rho = wc[0];
#pragma unroll
        for (int e = 1; e < NF; ++e) rho += wc[e];
        double G = eos.G_last, P = eos.P_last;
#pragma unroll
        for (int e = 0; e < I::NA; ++e) { G = fma(wc[I::A + e], eos.dG[e], G); P = fma(wc[I::A + e], eos.dP[e], P); }
        const double num = fma(G, wc[I::E], P) + wc[I::E];
        const double cs = sqrt(num / (G * rho));
#pragma unroll
        for (int d = 0; d < D; ++d) best = fmin(best, 1.0 / (g.inv_dx[d] * (fabs(wc[I::U + d]) + cs)));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) best = fmin(best, __shfl_xor_sync(0xffffffffu, best, off));
    __shared__ double red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int wi = 1; wi < (int)(blockDim.x >> 5); ++wi) best = fmin(best, red[wi]);
        atomicMin(min_bits, (unsigned long long)__double_as_longlong(best));
    }
}

// ---------------------------------------------------------------------------------------------------------
// a2 + a3 on one line of primitives (stage parity): same weno5 / hllc as the sweeps, one thread per cell.
// ---------------------------------------------------------------------------------------------------------
template <int D, int NF, int DIR>
__global__ void line_weno_kernel(Eos eos, int n, const double *__restrict__ w, double *vL, double *vR)
{
    using I = Idx<D, NF>;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;   // cell t - 1
    if (t >= n + 2) return;
    const int np = n + 2 * NG;
#pragma unroll
    for (int e = 0; e < I::NEQ; ++e) {
        const double *p = w + (long long)e * np + (t - 1 + NG);
        double l, r;
        weno5(p[0], p[-1] - p[-2], p[0] - p[-1], p[1] - p[0], p[2] - p[1], eos.weno_eps4, l, r);
        vL[(long long)e * (n + 2) + t] = l;
        vR[(long long)e * (n + 2) + t] = r;
    }
}

template <int D, int NF, int DIR>
__global__ void line_hllc_kernel(Eos eos, int n, const double *vL, const double *vR, double *F, double *uf)
{
    using I = Idx<D, NF>;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;   // face between cells t-1 and t
    if (t >= n + 1) return;
    double wl[I::NEQ], wr[I::NEQ], fl[I::NEQ], u;
#pragma unroll
    for (int e = 0; e < I::NEQ; ++e) { wl[e] = vL[(long long)e * (n + 2) + t]; wr[e] = vR[(long long)e * (n + 2) + t + 1]; }
    hllc<D, NF, DIR>(wl, wr, eos, fl, u);
#pragma unroll
    for (int e = 0; e < I::NEQ; ++e) F[(long long)e * (n + 1) + t] = fl[e];
    uf[t] = u;
}

}  // namespace mfc
