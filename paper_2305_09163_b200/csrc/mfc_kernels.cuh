// Kernels beside the fused right-hand side (mfc_fused.cuh): the CFL reduction and the stage-output kernels of
// the parity tests (cons->prim with ghost fill on the whole padded box; WENO5 + HLLC on one line).
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
// a6 CFL: dt = cfl * min over interior cells and directions of dx_d / (|u_d| + c)
//                          = cfl / max (|u_d| + c) / dx_d,
// so the kernel reduces the MAXIMUM of the signal speed over dx (no division per cell; the one reciprocal is
// taken on the host).  Non-negative doubles order like their bit patterns: the grid-wide maximum is an integer
// atomicMax.  Two cells per thread and trip keep twice the loads in flight (the kernel is HBM-bound: 56 B read
// per cell against about 70 FP64 instructions).
// ---------------------------------------------------------------------------------------------------------
template <int D, int NF>
__device__ __forceinline__ double cell_signal_speed(const double (&inv_dx)[3], const Eos &eos, const double (&qc)[2 * NF + D])
{
    using I = Idx<D, NF>;
    double wc[I::NEQ];
    cons_to_prim_cell<D, NF>(qc, eos, wc);
    double rho = wc[0];
#pragma unroll
    for (int e = 1; e < NF; ++e) rho += wc[e];
    double G = eos.G_last, P = eos.P_last;
#pragma unroll
    for (int e = 0; e < I::NA; ++e) { G = fma(wc[I::A + e], eos.dG[e], G); P = fma(wc[I::A + e], eos.dP[e], P); }
    const double num = fma(G, wc[I::E], P) + wc[I::E];               // (Gamma + 1) p + Pi
    const double cs = fabs(num) * rsqrt_fast(num * (G * rho));       // frozen mixture sound speed (reading B2)
    double s = 0.0, sum = 0.0;
#pragma unroll
    for (int d = 0; d < D; ++d) {
        const double sd = inv_dx[d] * (fabs(wc[I::U + d]) + cs);
        s = fmax(s, sd);
        sum += sd;                                                   // NaN if any direction is (fmax would drop it)
    }
    return sum == sum ? s : sum;
}

template <int D, int NF, bool NU>
__global__ void __launch_bounds__(256) cfl_kernel(typename GeoOf<NU>::type g, Eos eos, const double *__restrict__ q, unsigned long long *max_bits)
{
    using I = Idx<D, NF>;
    const long long ncell = (long long)g.n[0] * g.n[1] * g.n[2];
    const long long stride = (long long)gridDim.x * blockDim.x;
    // cell f of the interior (x fastest): offset in the padded array and the inverse widths of the cell (Eq. 8)
    auto cell_of = [&](long long f, double (&inv)[3]) -> long long {
        // (32-bit index arithmetic: 64-bit division costs more than the rest of the cell; the launcher checks the range)
        const unsigned fu = (unsigned)f, n0 = (unsigned)g.n[0], n1 = (unsigned)g.n[1];
        const unsigned r = fu / n0;
        const int i = (int)(fu - r * n0);
        const int k = (int)(r / n1), j = (int)(r - (unsigned)k * n1);
        if constexpr (NU) {
            inv[0] = __ldg(g.nu[0] + i + NG + 27 * g.nus[0]);
            inv[1] = D > 1 ? __ldg(g.nu[1] + j + NG + 27 * g.nus[1]) : 1.0;
            inv[2] = D > 2 ? __ldg(g.nu[2] + k + NG + 27 * g.nus[2]) : 1.0;
        } else {
            inv[0] = g.inv_dx[0]; inv[1] = g.inv_dx[1]; inv[2] = g.inv_dx[2];
        }
        return (long long)(k + g.g[2]) * g.sz + (long long)(j + g.g[1]) * g.sy + (i + NG);
    };
    // the maximum is taken on the BIT PATTERNS: non-negative doubles order like unsigned integers, and so do +inf and NaN
    // above them -- a non-finite signal speed (inadmissible state: negative c^2, rho = 0, NaN input) is not dropped the way
    // fmax would drop it, it wins the reduction and the host sees dt = NaN (mfc.h: inadmissible states propagate as NaN)
    unsigned long long best = 0ull;
    auto bits = [](double s) -> unsigned long long {
        return (unsigned long long)__double_as_longlong(s == s ? s : __longlong_as_double(0x7ff8000000000000ll));
    };
    for (long long f = (long long)blockIdx.x * blockDim.x + threadIdx.x; f < ncell; f += 2 * stride) {
        const bool two = f + stride < ncell;
        double i0[3], i1[3];
        const long long c0 = cell_of(f, i0), c1 = cell_of(two ? f + stride : f, i1);
        double q0[I::NEQ], q1[I::NEQ];
#pragma unroll
        for (int e = 0; e < I::NEQ; ++e) { q0[e] = __ldg(q + (long long)e * g.cells + c0); q1[e] = __ldg(q + (long long)e * g.cells + c1); }
        const unsigned long long b0 = bits(cell_signal_speed<D, NF>(i0, eos, q0)), b1 = bits(cell_signal_speed<D, NF>(i1, eos, q1));
        best = max(best, max(b0, b1));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, off));
    __shared__ unsigned long long red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int wi = 1; wi < (int)(blockDim.x >> 5); ++wi) best = max(best, red[wi]);
        atomicMax(max_bits, best);
    }
}

// ---------------------------------------------------------------------------------------------------------
// a2 + a3 on one line of primitives (stage parity): same weno5 / hllc as the sweeps, one thread per cell.
// ---------------------------------------------------------------------------------------------------------
template <int D, int NF, int DIR, int ORDER, bool NU>
__global__ void line_weno_kernel(Eos eos, int n, const double *__restrict__ w, double *vL, double *vR, const double *nu, int nus)
{
    using I = Idx<D, NF>;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;   // cell t - 1
    if (t >= n + 2) return;
    const int np = n + 2 * NG;
#pragma unroll
    for (int e = 0; e < I::NEQ; ++e) {
        const double *p = w + (long long)e * np + (t - 1 + NG);
        double l, r;
        reconstruct<ORDER, NU>(p[0], p[-1] - p[-2], p[0] - p[-1], p[1] - p[0], p[2] - p[1], eos.weno_eps4, l, r, NuRef{NU ? nu + t - 1 + NG : nullptr, nus});
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
