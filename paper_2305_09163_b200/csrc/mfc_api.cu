// C ABI of libmfc_b200 (include/mfc.h): context, scratch memory, the order of launches of one RHS evaluation
// and of the 3-stage TVD Runge-Kutta step, the CFL reduction, the host-buffer entry point and the
// measurement hooks.  No arithmetic of the method lives here: every step of the path runs in the kernels
// of mfc_kernels.cuh.  No CPU fallback.
#include "../../include/mfc.h"
#include "mfc_launch.h"
#include "mfc_math.cuh"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace mfc {

cudaError_t launch_prim(int ndim, int nf, const Geo &g, const Eos &e, const double *q, double *w, cudaStream_t s)
{
    switch (ndim) {
        case 1: return launch_prim_d1(nf, g, e, q, w, s);
        case 2: return launch_prim_d2(nf, g, e, q, w, s);
        case 3: return launch_prim_d3(nf, g, e, q, w, s);
    }
    return cudaErrorInvalidValue;
}
cudaError_t launch_rhs(int ndim, int nf, int order, const GeoNu &g, const Eos &e, const double *q, const SweepOut &o, int segment,
                       int path, cudaStream_t s)
{
    switch (ndim) {
        case 1: return launch_rhs_d1(nf, order, g, e, q, o, segment, path, s);
        case 2: return launch_rhs_d2(nf, order, g, e, q, o, segment, path, s);
        case 3: return launch_rhs_d3(nf, order, g, e, q, o, segment, path, s);
    }
    return cudaErrorInvalidValue;
}
cudaError_t launch_cfl(int ndim, int nf, const GeoNu &g, const Eos &e, const double *q, unsigned long long *min_bits,
                       cudaStream_t s)
{
    switch (ndim) {
        case 1: return launch_cfl_d1(nf, g, e, q, min_bits, s);
        case 2: return launch_cfl_d2(nf, g, e, q, min_bits, s);
        case 3: return launch_cfl_d3(nf, g, e, q, min_bits, s);
    }
    return cudaErrorInvalidValue;
}
cudaError_t launch_line(int ndim, int nf, int order, int dir, const Eos &e, int n, const double *w, double *vL, double *vR,
                        double *F, double *uf, const double *nu, int nus, cudaStream_t s)
{
    switch (ndim) {
        case 1: return launch_line_d1(nf, order, dir, e, n, w, vL, vR, F, uf, nu, nus, s);
        case 2: return launch_line_d2(nf, order, dir, e, n, w, vL, vR, F, uf, nu, nus, s);
        case 3: return launch_line_d3(nf, order, dir, e, n, w, vL, vR, F, uf, nu, nus, s);
    }
    return cudaErrorInvalidValue;
}

// ---------------------------------------------------------------------------------------------------------
// a0 ghost fill in memory ("buffers at the domain edges"): every ghost cell of the padded box takes the
// wrapped (periodic) or clamped (extrapolation) interior cell, dimension by dimension -- the index map composes, so
// one pass gives what filling x, then y, then z over the full padded extents gives, corners included.  Run before
// every evaluation of L: the TMA-staged march kernel then reads plain boxes of the padded array (a tile's halo is
// just the neighbouring cells, whatever the boundary kind).  One thread per ghost cell; the ghost shell is enumerated
// as the z slabs (full planes), the y slabs (full rows of the interior planes) and the x slabs (the rest).
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ghost_fill_kernel(Geo g, int neq, double *q)
{
    // (32-bit index arithmetic: the shell of any array that fits the device has fewer than 2^32 cells; checked by the launcher)
    const unsigned p0 = (unsigned)g.p[0], p1 = (unsigned)g.p[1], n1 = (unsigned)g.n[1];
    const unsigned nzs = (unsigned)(g.p[2] - g.n[2]) * p1 * p0;                      // z slabs: 2 g[2] planes
    const unsigned nys = (unsigned)g.n[2] * (unsigned)(g.p[1] - g.n[1]) * p0;        // y slabs: 2 g[1] rows per interior plane
    const unsigned nxs = (unsigned)g.n[2] * n1 * (unsigned)(g.p[0] - g.n[0]);        // x slabs: 2 g[0] cells per interior row
    const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    int i, j, k;
    if (t < nzs) {
        const unsigned r = t / p0;
        i = (int)(t - r * p0);
        const unsigned kk = r / p1;
        j = (int)(r - kk * p1);
        k = (int)kk < g.g[2] ? (int)kk : (int)kk + g.n[2];
    } else if (t < nzs + nys) {
        const unsigned u = t - nzs, r = u / p0, gy2 = 2u * (unsigned)g.g[1];
        i = (int)(u - r * p0);
        const unsigned kk = r / gy2, jj = r - kk * gy2;
        j = (int)jj < g.g[1] ? (int)jj : (int)jj + g.n[1];
        k = (int)kk + g.g[2];
    } else if (t < nzs + nys + nxs) {
        const unsigned u = t - nzs - nys, gx2 = 2u * (unsigned)g.g[0], r = u / gx2, ii = u - r * gx2;
        i = (int)ii < g.g[0] ? (int)ii : (int)ii + g.n[0];
        const unsigned kk = r / n1;
        j = (int)(r - kk * n1) + g.g[1];
        k = (int)kk + g.g[2];
    } else return;
    const int si = bc_source(i - g.g[0], g.n[0], g.bc_lo[0], g.bc_hi[0]) + g.g[0];
    const int sj = bc_source(j - g.g[1], g.n[1], g.bc_lo[1], g.bc_hi[1]) + g.g[1];
    const int sk = bc_source(k - g.g[2], g.n[2], g.bc_lo[2], g.bc_hi[2]) + g.g[2];
    const long long dst = (long long)k * g.sz + (long long)j * g.sy + i;
    const long long src = (long long)sk * g.sz + (long long)sj * g.sy + si;
    if (src == dst) return;     // a ghost cell of a HALO side in every dimension it is a ghost of: the caller's, left alone
    for (int e = 0; e < neq; ++e) q[(long long)e * g.cells + dst] = q[(long long)e * g.cells + src];
}

cudaError_t launch_ghost_fill(const Geo &g, int neq, double *q, cudaStream_t s)
{
    const long long shell = g.cells - (long long)g.n[0] * g.n[1] * g.n[2];
    if (shell <= 0) return cudaSuccess;
    if (shell >= (1ll << 32) - 256) return cudaErrorInvalidValue;
    ghost_fill_kernel<<<(unsigned)((shell + 255) / 256), 256, 0, s>>>(g, neq, q);
    return cudaGetLastError();
}

__global__ void eos_seed_kernel(const double *gm1, double *ygm1, int n)
{
    if ((int)threadIdx.x < n) ygm1[threadIdx.x] = div_seed(gm1[threadIdx.x]);
}
cudaError_t launch_eos_seed(const double *gm1_dev, double *ygm1_dev, int n, cudaStream_t s)
{
    eos_seed_kernel<<<1, 32, 0, s>>>(gm1_dev, ygm1_dev, n);
    return cudaGetLastError();
}

struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

struct EventPair {
    cudaEvent_t a, b;
    int kid;
};

}  // namespace mfc

struct mfc_ctx {
    int ndim = 0, nf = 0, neq = 0, device = 0, segment = 0, order = 5, staging = 0;
    double cfl = 0.3;
    long long elems = 0;
    mfc::GeoNu g{};
    mfc::Eos e{};
    double *q1 = nullptr, *q2 = nullptr, *q_own = nullptr;
    double *nu_dev[3] = {nullptr, nullptr, nullptr};   // non-uniform spacing: per-direction coefficient tables
    unsigned long long *min_dev = nullptr;
    unsigned long long *min_host = nullptr;  // pinned
    cudaEvent_t dt_ready = nullptr;          // recorded behind the copy of the reduction's result: the host waits for it alone
    bool profile = false;
    std::vector<mfc::EventPair> pending;
    std::vector<cudaEvent_t> pool;
    double ms[MFC_K_COUNT] = {0, 0, 0, 0};
    long long launches[MFC_K_COUNT] = {0, 0, 0, 0};
    long long launch_total = 0;
    cudaError_t last_cuda = cudaSuccess;     // the CUDA error behind the last MFC_ECUDA / MFC_ENOMEM of this context
};

namespace {

using namespace mfc;

int flush_events(mfc_ctx *c)
{
    for (auto &p : c->pending) {
        if (cudaEventSynchronize(p.b) != cudaSuccess) return MFC_ECUDA;
        float t = 0.f;
        if (cudaEventElapsedTime(&t, p.a, p.b) != cudaSuccess) return MFC_ECUDA;
        c->ms[p.kid] += (double)t;
        c->pool.push_back(p.a);
        c->pool.push_back(p.b);
    }
    c->pending.clear();
    return MFC_OK;
}

cudaEvent_t get_event(mfc_ctx *c)
{
    if (!c->pool.empty()) {
        cudaEvent_t e = c->pool.back();
        c->pool.pop_back();
        return e;
    }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}

// brackets one kernel launch with events when profiling is on, and counts it
struct Timed {
    mfc_ctx *c;
    int kid;
    cudaStream_t s;
    cudaEvent_t a = nullptr, b = nullptr;
    Timed(mfc_ctx *c_, int kid_, cudaStream_t s_) : c(c_), kid(kid_), s(s_)
    {
        if (c->profile) {
            if (c->pending.size() >= 8192) flush_events(c);
            a = get_event(c);
            b = get_event(c);
            cudaEventRecord(a, s);
        }
    }
    ~Timed()
    {
        c->launches[kid] += 1;
        c->launch_total += 1;
        if (a) {
            cudaEventRecord(b, s);
            c->pending.push_back({a, b, kid});
        }
    }
};

int cuda_to_status(cudaError_t e, mfc_ctx *c = nullptr)
{
    if (e == cudaSuccess) return MFC_OK;
    if (c) c->last_cuda = e;
    if (e == cudaErrorMemoryAllocation) return MFC_ENOMEM;
    return MFC_ECUDA;
}

// One evaluation of L(q_in): the ghost cells of q_in are filled in memory (a0), then one launch computes
// out = base + coef L(q_in), base described by `o` (SweepOut, mfc_launch.h).
int fill_ghosts_of(mfc_ctx *c, double *q_in, cudaStream_t s)
{
    bool all_halo = true;
    for (int d = 0; d < c->ndim; ++d) all_halo = all_halo && c->g.bc_lo[d] == MFC_BC_HALO && c->g.bc_hi[d] == MFC_BC_HALO;
    if (all_halo) return MFC_OK;
    Timed t(c, MFC_K_GHOST, s);
    return cuda_to_status(launch_ghost_fill(c->g, c->neq, q_in, s), c);
}
int eval_L(mfc_ctx *c, double *q_in, const SweepOut &o, cudaStream_t s, bool ghosts_filled = false)
{
    if (!ghosts_filled) {
        const int st = fill_ghosts_of(c, q_in, s);
        if (st) return st;
    }
    cudaError_t err = cudaSuccess;
    {
        Timed t(c, MFC_K_RHS, s);
        err = launch_rhs(c->ndim, c->nf, c->order, c->g, c->e, q_in, o, c->segment, c->staging, s);
    }
    return cuda_to_status(err, c);
}

// 3-stage TVD Runge-Kutta.  Every stage is out = ca qn + cb (qs + dt L(qs)).  A stage reads its
// neighbours' cells of qs, so it never writes the array it evaluates L on: q -> q1 -> q2 -> q.
int rk3_stage(mfc_ctx *c, int stage, double *q, double dt, cudaStream_t s, bool ghosts_filled = false)
{
    SweepOut f{};
    switch (stage) {
        case 0:   // q1 = q + dt L(q)
            f.out = c->q1; f.qs = q; f.qn = q; f.ca = 0.0; f.cb = 1.0; f.coef = dt; f.nbase = 1;
            return eval_L(c, q, f, s, ghosts_filled);
        case 1:   // q2 = 3/4 q + 1/4 (q1 + dt L(q1))
            f.out = c->q2; f.qs = c->q1; f.qn = q; f.ca = 0.75; f.cb = 0.25; f.coef = 0.25 * dt; f.nbase = 2;
            return eval_L(c, c->q1, f, s);
        case 2:   // q <- 1/3 q + 2/3 (q2 + dt L(q2))
            f.out = q; f.qs = c->q2; f.qn = q; f.ca = 1.0 / 3.0; f.cb = 2.0 / 3.0; f.coef = (2.0 / 3.0) * dt; f.nbase = 2;
            return eval_L(c, c->q2, f, s);
    }
    return MFC_EINVAL;
}

int rk3(mfc_ctx *c, double *q, double dt, cudaStream_t s)
{
    for (int stage = 0; stage < 3; ++stage) {
        const int st = rk3_stage(c, stage, q, dt, s);
        if (st) return st;
    }
    return MFC_OK;
}

// the reduction and the copy of its result, enqueued; cfl_dt_finish waits for them
int cfl_dt_enqueue(mfc_ctx *c, const double *q, cudaStream_t s)
{
    cudaError_t err = cudaMemsetAsync(c->min_dev, 0, sizeof(unsigned long long), s);   // max of speeds / dx
    if (err != cudaSuccess) return cuda_to_status(err, c);
    {
        Timed t(c, MFC_K_CFL, s);
        err = launch_cfl(c->ndim, c->nf, c->g, c->e, q, c->min_dev, s);
    }
    if (err != cudaSuccess) return cuda_to_status(err, c);
    err = cudaMemcpyAsync(c->min_host, c->min_dev, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s);
    if (err == cudaSuccess) err = cudaEventRecord(c->dt_ready, s);
    return cuda_to_status(err, c);
}
// waits for the copy only (not for work enqueued behind it)
int cfl_dt_finish(mfc_ctx *c, double *dt_host)
{
    const cudaError_t err = cudaEventSynchronize(c->dt_ready);
    if (err != cudaSuccess) return cuda_to_status(err, c);
    double v;
    std::memcpy(&v, c->min_host, sizeof(double));
    *dt_host = c->cfl * (1.0 / v);   // v = max over cells and directions of (|u_d| + c) / dx_d
    return MFC_OK;
}

// One step at the CFL time step of the current state (a6 then a0 - a5, three times).  The host needs dt before it can launch
// the first stage (dt is a kernel argument), so every step has one device -> host round trip; the ghost fill of stage 0
// does not depend on dt and is enqueued BEFORE the wait, so the device works through the round trip instead of idling.
int step_cfl(mfc_ctx *c, double *q, double *dt_out, cudaStream_t s)
{
    int st = cfl_dt_enqueue(c, q, s);
    if (st) return st;
    st = fill_ghosts_of(c, q, s);
    if (st) return st;
    double dt = 0.0;
    st = cfl_dt_finish(c, &dt);
    if (st) return st;
    if (dt_out) *dt_out = dt;
    if (!std::isfinite(dt) || !(dt > 0.0)) return MFC_ENONFINITE;    // inadmissible state: do not step on
    for (int stage = 0; stage < 3; ++stage) {
        st = rk3_stage(c, stage, q, dt, s, stage == 0);
        if (st) return st;
    }
    return MFC_OK;
}

int cfl_dt(mfc_ctx *c, const double *q, double *dt_host, cudaStream_t s)
{
    const int st = cfl_dt_enqueue(c, q, s);
    return st ? st : cfl_dt_finish(c, dt_host);
}

// FP64 FMA micro-benchmark: 8 independent register-resident DFMA chains per thread.  Two operand shapes, the faster one
// counts: V = 0  x = fma(x, m, a) with m and a in registers (three distinct 64-bit register operands: 92 % of the FP64 pipe,
// measured with ncu -- operand fetch, not the pipe, is what saturates);  V = 1  x = fma(x, m, x) with m a kernel parameter
// (constant bank): one register pair per instruction.
template <int V>
__global__ void __launch_bounds__(256) dfma_probe_kernel(double *out, int iters, double m, double a)
{
    double x0 = 1.0 + threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if constexpr (V == 0) {
                x0 = fma(x0, m, a); x1 = fma(x1, m, a); x2 = fma(x2, m, a); x3 = fma(x3, m, a);
                x4 = fma(x4, m, a); x5 = fma(x5, m, a); x6 = fma(x6, m, a); x7 = fma(x7, m, a);
            } else {
                x0 = fma(x0, m, x0); x1 = fma(x1, m, x1); x2 = fma(x2, m, x2); x3 = fma(x3, m, x3);
                x4 = fma(x4, m, x4); x5 = fma(x5, m, x5); x6 = fma(x6, m, x6); x7 = fma(x7, m, x7);
            }
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}


// ---------------------------------------------------------------------------------------------------------
// Non-uniform spacing: the per-index coefficient tables of Listing 1 (poly_coef, beta_coef, d_cb), built
// once per context on the host.  The reconstruction polynomial of a stencil is the derivative of the Newton interpolant
// (divided differences) of the primitive function of the cell averages at the stencil's edges (refs. [17], [38]); every
// table entry is that polynomial, or one of its derivatives, applied to a unit datum.
// ---------------------------------------------------------------------------------------------------------
// d^k/dx^k at x (k = 1, 2, 3) of the Newton interpolant of V(e_m) = sum_{l < m} u_l (e_{l+1} - e_l), nc cells, nc + 1 edges
double newton_primitive_deriv(const double *e, int nc, const double *u, double x, int k)
{
    double dd[8];
    dd[0] = 0.0;
    for (int m = 1; m <= nc; ++m) dd[m] = dd[m - 1] + u[m - 1] * (e[m] - e[m - 1]);
    for (int lev = 1; lev <= nc; ++lev)
        for (int m = nc; m >= lev; --m) dd[m] = (dd[m] - dd[m - 1]) / (e[m] - e[m - lev]);
    // omega_m = prod_{l < m} (x - e_l) and its first three derivatives, by the product rule
    double w0 = 1.0, w1 = 0.0, w2 = 0.0, w3 = 0.0, res = 0.0;
    for (int m = 0; m <= nc; ++m) {
        res += dd[m] * (k == 1 ? w1 : (k == 2 ? w2 : w3));
        const double f = x - e[m];
        w3 = w3 * f + 3.0 * w2;
        w2 = w2 * f + 2.0 * w1;
        w1 = w1 * f + w0;
        w0 = w0 * f;
    }
    return res;
}

// padded edges from the interior ones: a ghost cell has the width of the cell its value comes from (mfc.h)
std::vector<double> padded_edges(const double *edges, int n, int bc_lo, int bc_hi)
{
    std::vector<double> xe(n + 2 * NG + 1);
    for (int i = 0; i <= n; ++i) xe[NG + i] = edges[i];
    for (int m = 1; m <= NG; ++m) {
        const int sl = bc_lo == MFC_BC_PERIODIC ? n - m : 0;            // interior cell the ghost cell -m copies
        const int sh = bc_hi == MFC_BC_PERIODIC ? m - 1 : n - 1;        // ... and the ghost cell n - 1 + m
        xe[NG - m] = xe[NG - m + 1] - (edges[sl + 1] - edges[sl]);
        xe[NG + n + m] = xe[NG + n + m - 1] + (edges[sh + 1] - edges[sh]);
    }
    return xe;
}

// table [NU_NC][stride] of one direction; false if an ideal weight is not positive
bool nu_tables(const std::vector<double> &xe, int p, int stride, std::vector<double> &tab)
{
    tab.assign((size_t)NU_NC * stride, 0.0);
    bool ok = true;
    for (int j = 2; j <= p - 3; ++j) {
        const double xm = xe[j], xp = xe[j + 1], h = xp - xm, xc = 0.5 * (xm + xp);
        double *t = tab.data() + j;
        auto put = [&](int k, double v) { t[(size_t)k * stride] = v; };
        double dL[3], dR[3], pL[3][2], pR[3][2];
        const double e5[5][5] = {{1, 0, 0, 0, 0}, {0, 1, 0, 0, 0}, {0, 0, 1, 0, 0}, {0, 0, 0, 1, 0}, {0, 0, 0, 0, 1}};
        for (int r = 0; r < 3; ++r) {
            const double *e = &xe[j - 2 + r];
            const int lc = 2 - r;                                       // the centre cell within the stencil
            const double uA[3] = {0, 1, 1}, uB[3] = {0, 0, 1};          // unit differences: (d1, d2) = (1, 0) and (0, 1)
            pL[r][0] = newton_primitive_deriv(e, 3, uA, xp, 1) - uA[lc];
            pL[r][1] = newton_primitive_deriv(e, 3, uB, xp, 1) - uB[lc];
            pR[r][0] = newton_primitive_deriv(e, 3, uA, xm, 1) - uA[lc];
            pR[r][1] = newton_primitive_deriv(e, 3, uB, xm, 1) - uB[lc];
            // p_r = a0 + a1 (x - xc) + a2 (x - xc)^2:  a1 = p'(xc), a2 = p'' / 2;  beta = a1^2 h^2 + 13/3 a2^2 h^4 (Jiang-Shu)
            const double l1 = newton_primitive_deriv(e, 3, uA, xc, 2), l2 = newton_primitive_deriv(e, 3, uB, xc, 2);
            const double m1 = 0.5 * newton_primitive_deriv(e, 3, uA, xc, 3), m2 = 0.5 * newton_primitive_deriv(e, 3, uB, xc, 3);
            const double h2 = h * h, h4 = h2 * h2;
            put(3 * r + 0, h2 * l1 * l1 + 13.0 / 3.0 * h4 * m1 * m1);
            put(3 * r + 1, 2.0 * h2 * l1 * l2 + 26.0 / 3.0 * h4 * m1 * m2);
            put(3 * r + 2, h2 * l2 * l2 + 13.0 / 3.0 * h4 * m2 * m2);
        }
        // ideal weights: the combination of the three quadratics that equals the five-cell quartic at the face; the outermost
        // cells belong to one stencil each
        const double *e5e = &xe[j - 2];
        const double u3first[3] = {1, 0, 0}, u3last[3] = {0, 0, 1};
        for (int side = 0; side < 2; ++side) {
            const double x = side == 0 ? xp : xm;
            double *d = side == 0 ? dL : dR;
            d[0] = newton_primitive_deriv(e5e, 5, e5[0], x, 1) / newton_primitive_deriv(&xe[j - 2], 3, u3first, x, 1);
            d[2] = newton_primitive_deriv(e5e, 5, e5[4], x, 1) / newton_primitive_deriv(&xe[j], 3, u3last, x, 1);
            d[1] = 1.0 - d[0] - d[2];
            for (int r = 0; r < 3; ++r) ok = ok && d[r] > 0.0;
        }
        for (int r = 0; r < 3; ++r) {
            put(9 + 2 * r, dL[r] * pL[r][0]);
            put(10 + 2 * r, dL[r] * pL[r][1]);
            put(15 + 2 * r, dR[r] * pR[r][0]);
            put(16 + 2 * r, dR[r] * pR[r][1]);
            put(21 + r, dL[r]);
            put(24 + r, dR[r]);
        }
        put(27, 1.0 / h);
    }
    // entries without a full stencil and the padding past the last cell: copies of the nearest valid cell (read by threads
    // that write nothing, never used)
    for (int k = 0; k < NU_NC; ++k) {
        double *row = tab.data() + (size_t)k * stride;
        for (int j = 0; j < 2 && j < stride; ++j) row[j] = row[2];
        for (int j = p - 2; j < stride; ++j) row[j] = row[p - 3];
    }
    return ok;
}

}  // namespace

extern "C" {

const char *mfc_strerror(int code)
{
    switch (code) {
        case MFC_OK: return "ok";
        case MFC_EINVAL: return "invalid argument";
        case MFC_EUNSUPPORTED: return "(ndim, n_fluids) not in the compiled template set";
        case MFC_ECUDA: return "CUDA runtime error";
        case MFC_ENOMEM: return "out of memory";
        case MFC_ENONFINITE: return "the state is not admissible: the CFL time step is not finite";
        case MFC_ELIMIT: return "grid too large for the fixed workspace of mfc_cfl_dt_static (MFC_STATIC_MAX_CELLS interior cells)";
    }
    return "unknown error";
}

const char *mfc_version(void) { return "mfc-b200 0.3 (sm_100a)"; }

int mfc_abi_version(void) { return MFC_ABI_VERSION; }

const char *mfc_cuda_error(const mfc_ctx *c) { return c ? cudaGetErrorString(c->last_cuda) : "no context"; }

int mfc_init(mfc_ctx **out, const mfc_grid *grid, int n_fluids, const mfc_fluid *eos, const mfc_bc *bc, const mfc_opts *opts)
{
    if (!out || !grid || !eos || !bc) return MFC_EINVAL;
    *out = nullptr;
    if (opts && opts->abi_version != 0 && opts->abi_version != MFC_ABI_VERSION) return MFC_EINVAL;   // header / library mismatch
    if (grid->ndim < 1 || grid->ndim > 3 || n_fluids < 1) return MFC_EINVAL;
    if (n_fluids > MFC_MAX_FLUIDS) return MFC_EUNSUPPORTED;
    if (opts && opts->kapila && n_fluids != 2) return MFC_EUNSUPPORTED;
    const int order = (opts && opts->weno_order != 0) ? opts->weno_order : 5;
    if (order != 1 && order != 3 && order != 5) return MFC_EINVAL;
    if (opts && (opts->staging < 0 || opts->staging > 3)) return MFC_EINVAL;
    bool nonuniform = false;
    for (int d = 0; d < grid->ndim; ++d) {
        if (grid->n[d] < MFC_NG) return MFC_EINVAL;
        if (grid->edges_host[d]) {
            // the widths of HALO ghost cells are the neighbour's: not expressible through edges_host yet
            if (bc->lo[d] == MFC_BC_HALO || bc->hi[d] == MFC_BC_HALO) return MFC_EUNSUPPORTED;
            nonuniform = true;
            for (int i = 0; i < grid->n[d]; ++i)
                if (!(grid->edges_host[d][i + 1] > grid->edges_host[d][i]) || !std::isfinite(grid->edges_host[d][i + 1] - grid->edges_host[d][i])) return MFC_EINVAL;
        } else if (!(grid->hi[d] > grid->lo[d])) return MFC_EINVAL;
        if (grid->inv_dx[d] != 0.0 && (grid->edges_host[d] || !(grid->inv_dx[d] > 0.0) || !std::isfinite(grid->inv_dx[d]))) return MFC_EINVAL;
        if (bc->lo[d] < MFC_BC_PERIODIC || bc->lo[d] > MFC_BC_HALO) return MFC_EINVAL;
        if (bc->hi[d] < MFC_BC_PERIODIC || bc->hi[d] > MFC_BC_HALO) return MFC_EINVAL;
        if ((bc->lo[d] == MFC_BC_PERIODIC) != (bc->hi[d] == MFC_BC_PERIODIC)) return MFC_EINVAL;
    }
    if (nonuniform && order != 5) return MFC_EUNSUPPORTED;
    for (int i = 0; i < n_fluids; ++i)
        if (!(eos[i].gamma > 1.0) || !std::isfinite(eos[i].gamma) || !std::isfinite(eos[i].pi_inf)) return MFC_EINVAL;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return MFC_ECUDA;
    int dev = opts ? opts->device : -1;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return MFC_ECUDA;
    if (dev >= ndev) return MFC_EINVAL;

    mfc_ctx *c = new (std::nothrow) mfc_ctx();
    if (!c) return MFC_ENOMEM;
    c->ndim = grid->ndim;
    c->nf = n_fluids;
    c->neq = 2 * n_fluids + grid->ndim;
    c->device = dev;
    c->cfl = (opts && opts->cfl > 0.0) ? opts->cfl : 0.3;
    c->order = order;
    const double eps = (opts && opts->weno_eps > 0.0) ? opts->weno_eps : 1.0e-16;

    GeoNu &g = c->g;
    g.ndim = grid->ndim;
    for (int d = 0; d < 3; ++d) {
        const bool act = d < grid->ndim;
        g.n[d] = act ? grid->n[d] : 1;
        g.g[d] = act ? NG : 0;
        g.p[d] = g.n[d] + 2 * g.g[d];
        g.inv_dx[d] = act && !grid->edges_host[d] ? (grid->inv_dx[d] > 0.0 ? grid->inv_dx[d] : (double)grid->n[d] / (grid->hi[d] - grid->lo[d])) : 1.0;
        g.bc_lo[d] = act ? bc->lo[d] : MFC_BC_EXTRAP;
        g.bc_hi[d] = act ? bc->hi[d] : MFC_BC_EXTRAP;
    }
    g.sy = g.p[0];
    g.sz = (long long)g.p[0] * g.p[1];
    g.cells = g.sz * g.p[2];
    c->elems = g.cells * c->neq;

    Eos &e = c->e;
    std::memset(&e, 0, sizeof(e));
    double Gm[MAX_NF], Pm[MAX_NF];
    for (int i = 0; i < n_fluids; ++i) {
        e.gamma[i] = eos[i].gamma;
        e.pi_inf[i] = eos[i].pi_inf;
        e.gm1[i] = eos[i].gamma - 1.0;
        Gm[i] = 1.0 / (eos[i].gamma - 1.0);
        Pm[i] = eos[i].gamma * eos[i].pi_inf / (eos[i].gamma - 1.0);
    }
    e.G_last = Gm[n_fluids - 1];
    e.P_last = Pm[n_fluids - 1];
    for (int i = 0; i < n_fluids - 1; ++i) {
        e.dG[i] = Gm[i] - e.G_last;
        e.dP[i] = Pm[i] - e.P_last;
    }
    e.weno_eps4 = 4.0 * eps;
    e.kapila = (opts && opts->kapila) ? 1 : 0;

    c->segment = (opts && opts->march_segment > 0) ? opts->march_segment : 0;   // 0: the launcher's heuristic
    c->staging = opts ? opts->staging : 0;

    DeviceGuard guard(dev);
    if (cudaDeviceGetAttribute(&g.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) g.sms = 0;
    const size_t bytes = (size_t)c->elems * sizeof(double);
    cudaError_t err = cudaMalloc((void **)&c->q1, bytes);
    if (err == cudaSuccess) err = cudaMalloc((void **)&c->q2, bytes);
    if (err == cudaSuccess) err = cudaMalloc((void **)&c->min_dev, sizeof(unsigned long long));
    if (err == cudaSuccess) err = cudaMallocHost((void **)&c->min_host, sizeof(unsigned long long));
    if (err == cudaSuccess) err = cudaEventCreateWithFlags(&c->dt_ready, cudaEventDisableTiming);
    if (err == cudaSuccess) {   // reciprocal seeds of gamma_i - 1, as the device computes them (mfc_math.cuh div_seed)
        double *tmp = nullptr;
        err = cudaMalloc((void **)&tmp, 2 * MAX_NF * sizeof(double));
        if (err == cudaSuccess) err = cudaMemcpy(tmp, e.gm1, MAX_NF * sizeof(double), cudaMemcpyHostToDevice);
        if (err == cudaSuccess) err = launch_eos_seed(tmp, tmp + MAX_NF, n_fluids, 0);
        if (err == cudaSuccess) err = cudaMemcpy(e.ygm1, tmp + MAX_NF, MAX_NF * sizeof(double), cudaMemcpyDeviceToHost);
        cudaFree(tmp);
    }
    // non-uniform spacing: coefficient tables of every active dimension (a uniform dimension of a mixed grid gets the
    // tables of its uniform edges), rows padded so that ragged tiles read defined entries
    for (int d = 0; d < 3; ++d) { g.nu[d] = nullptr; g.nus[d] = 0; }
    if (err == cudaSuccess && nonuniform) {
        for (int d = 0; d < grid->ndim && err == cudaSuccess; ++d) {
            std::vector<double> uni;
            const double *edges = grid->edges_host[d];
            if (!edges) {
                uni.resize(grid->n[d] + 1);
                for (int i = 0; i <= grid->n[d]; ++i) uni[i] = grid->lo[d] + (grid->hi[d] - grid->lo[d]) * ((double)i / grid->n[d]);
                edges = uni.data();
            }
            const std::vector<double> xe = padded_edges(edges, grid->n[d], bc->lo[d], bc->hi[d]);
            std::vector<double> tab;
            g.nus[d] = g.p[d] + 64;
            if (!nu_tables(xe, g.p[d], g.nus[d], tab)) {
                mfc_destroy(c);
                return MFC_EUNSUPPORTED;
            }
            err = cudaMalloc((void **)&c->nu_dev[d], tab.size() * sizeof(double));
            if (err == cudaSuccess) err = cudaMemcpy(c->nu_dev[d], tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice);
            g.nu[d] = c->nu_dev[d];
        }
    }
    if (err != cudaSuccess) {
        const int st = cuda_to_status(err);
        cudaGetLastError();
        mfc_destroy(c);
        return st;
    }
    *out = c;
    return MFC_OK;
}

void mfc_destroy(mfc_ctx *c)
{
    if (!c) return;
    {
        DeviceGuard guard(c->device);
        flush_events(c);
        for (cudaEvent_t ev : c->pool) cudaEventDestroy(ev);
        cudaFree(c->q1);
        cudaFree(c->q2);
        cudaFree(c->q_own);
        for (int d = 0; d < 3; ++d) cudaFree(c->nu_dev[d]);
        cudaFree(c->min_dev);
        if (c->min_host) cudaFreeHost(c->min_host);
        if (c->dt_ready) cudaEventDestroy(c->dt_ready);
    }
    delete c;
}

int mfc_layout(const mfc_ctx *c, int *neq, int *ng, long long padded_n[3], long long *elems)
{
    if (!c) return MFC_EINVAL;
    if (neq) *neq = c->neq;
    if (ng) *ng = MFC_NG;
    if (padded_n)
        for (int d = 0; d < 3; ++d) padded_n[d] = c->g.p[d];
    if (elems) *elems = c->elems;
    return MFC_OK;
}

int mfc_rhs(mfc_ctx *c, double *q_dev, double *rhs_dev, void *stream)
{
    if (!c || !q_dev || !rhs_dev || q_dev == rhs_dev) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    SweepOut f{};
    f.out = rhs_dev; f.coef = 1.0; f.nbase = 0;
    return eval_L(c, q_dev, f, (cudaStream_t)stream);
}

int mfc_rk3_step(mfc_ctx *c, double *q_dev, double dt, void *stream)
{
    if (!c || !q_dev) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    return rk3(c, q_dev, dt, (cudaStream_t)stream);
}

int mfc_rk3_stage(mfc_ctx *c, int stage, double *q_dev, double dt, void *stream)
{
    if (!c || !q_dev || stage < 0 || stage > 2) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    return rk3_stage(c, stage, q_dev, dt, (cudaStream_t)stream);
}

int mfc_stage_array(mfc_ctx *c, int k, double **array_dev)
{
    if (!c || !array_dev || (k != 1 && k != 2)) return MFC_EINVAL;
    *array_dev = k == 1 ? c->q1 : c->q2;
    return MFC_OK;
}

int mfc_step_cfl(mfc_ctx *c, double *q_dev, double *dt_host, void *stream)
{
    if (!c || !q_dev) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    return step_cfl(c, q_dev, dt_host, (cudaStream_t)stream);
}

int mfc_cfl_dt(mfc_ctx *c, const double *q_dev, double *dt_host, void *stream)
{
    if (!c || !q_dev || !dt_host) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    return cfl_dt(c, q_dev, dt_host, (cudaStream_t)stream);
}

int mfc_advance_host(mfc_ctx *c, double *q_host, int nsteps, double dt_fixed, double *t_host, void *stream)
{
    if (!c || !q_host || nsteps < 0) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t bytes = (size_t)c->elems * sizeof(double);
    if (!c->q_own) {
        cudaError_t err = cudaMalloc((void **)&c->q_own, bytes);
        if (err != cudaSuccess) {
            cudaGetLastError();
            return cuda_to_status(err, c);
        }
    }
    cudaError_t cerr = cudaMemcpyAsync(c->q_own, q_host, bytes, cudaMemcpyHostToDevice, s);
    if (cerr != cudaSuccess) return cuda_to_status(cerr, c);
    double t = 0.0;
    for (int it = 0; it < nsteps; ++it) {
        double dt = dt_fixed;
        const int st = dt_fixed > 0.0 ? rk3(c, c->q_own, dt, s) : step_cfl(c, c->q_own, &dt, s);
        if (st) return st;                                           // (MFC_ENONFINITE: the step was not taken)
        t += dt;
    }
    cerr = cudaMemcpyAsync(q_host, c->q_own, bytes, cudaMemcpyDeviceToHost, s);
    if (cerr == cudaSuccess) cerr = cudaStreamSynchronize(s);
    if (cerr != cudaSuccess) return cuda_to_status(cerr, c);
    if (t_host) *t_host = t;
    return MFC_OK;
}

int mfc_cons_to_prim(mfc_ctx *c, const double *q_dev, double *w_dev, void *stream)
{
    if (!c || !q_dev || !w_dev || q_dev == w_dev) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    cudaError_t err;
    {
        Timed t(c, MFC_K_PRIM, (cudaStream_t)stream);
        err = launch_prim(c->ndim, c->nf, c->g, c->e, q_dev, w_dev, (cudaStream_t)stream);
    }
    return cuda_to_status(err, c);
}

int mfc_line_fluxes(mfc_ctx *c, int dir, int n, const double *w_dev, double *vL_dev, double *vR_dev, double *F_dev,
                    double *uface_dev, void *stream)
{
    if (!c || !w_dev || !vL_dev || !vR_dev || !F_dev || !uface_dev || n < 1 || dir < 0 || dir >= c->ndim) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    if (c->g.nu[0] && n != c->g.n[dir]) return MFC_EINVAL;     // the tables are those of the grid's own lines
    c->launch_total += 2;                                      // (a refused call launches nothing)
    return cuda_to_status(launch_line(c->ndim, c->nf, c->order, dir, c->e, n, w_dev, vL_dev, vR_dev, F_dev, uface_dev, c->g.nu[dir], c->g.nus[dir],
                                      (cudaStream_t)stream), c);
}

int mfc_profile_enable(mfc_ctx *c, int on)
{
    if (!c) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    if (!on) {
        const int st = flush_events(c);
        if (st) return st;
    }
    c->profile = on != 0;
    return MFC_OK;
}

int mfc_profile_get(mfc_ctx *c, int kernel_id, long long *launches, double *total_ms, int reset)
{
    if (!c || kernel_id < 0 || kernel_id >= MFC_K_COUNT) return MFC_EINVAL;
    DeviceGuard guard(c->device);
    const int st = flush_events(c);
    if (st) return st;
    if (launches) *launches = c->launches[kernel_id];
    if (total_ms) *total_ms = c->ms[kernel_id];
    if (reset) {
        c->launches[kernel_id] = 0;
        c->ms[kernel_id] = 0.0;
    }
    return MFC_OK;
}

long long mfc_launch_count(const mfc_ctx *c) { return c ? c->launch_total : 0; }

int mfc_probe_dfma(int device, double *tflops_host, double *ms_host)
{
    if (!tflops_host) return MFC_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return MFC_ECUDA;
    if (device < 0 && cudaGetDevice(&device) != cudaSuccess) return MFC_ECUDA;
    if (device >= ndev) return MFC_EINVAL;
    DeviceGuard guard(device);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return MFC_ECUDA;
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 4096;
    double *out = nullptr;
    if (cudaMalloc((void **)&out, sizeof(double) * (size_t)blocks * threads) != cudaSuccess) return MFC_ENOMEM;
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    float best = 1e30f;
    for (int variant = 0; variant < 2; ++variant) {
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(a, 0);
            if (variant == 0) dfma_probe_kernel<0><<<blocks, threads>>>(out, iters, 1.0 - 1e-9, 1e-9);
            else dfma_probe_kernel<1><<<blocks, threads>>>(out, iters, -1e-9, 0.0);
            cudaEventRecord(b, 0);
            cudaEventSynchronize(b);
            float t = 0.f;
            cudaEventElapsedTime(&t, a, b);
            if (rep > 0 && t < best) best = t;
        }
    }
    const cudaError_t err = cudaGetLastError();
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(out);
    if (err != cudaSuccess) return MFC_ECUDA;
    const double flops = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads;
    *tflops_host = flops / ((double)best * 1e-3) / 1e12;
    if (ms_host) *ms_host = (double)best;
    return MFC_OK;
}

}  // extern "C"
