// Host-side description of one launch of each kernel family.  Plain structs passed by value to the kernels;
// the per-dimension translation units (mfc_inst_d{1,2,3}.cu) implement the launchers declared at the end.
#pragma once
#include <cuda_runtime.h>

namespace mfc {

constexpr int NG = 3;        // ghost layers, PAPER.md:168 (WENO5 stencil)
constexpr int MAX_NF = 3;

// padded box, x fastest (Listing 1 index order)
struct Geo {
    int ndim;
    int n[3];            // interior cells (1 in inactive dimensions)
    int p[3];            // padded extents (n + 2 NG in active dimensions, else 1)
    int g[3];            // ghost offset per dimension (NG if active, else 0)
    long long sy, sz;    // strides of y and z in cells (sx = 1)
    long long cells;     // p[0] * p[1] * p[2] : stride between equations
    double inv_dx[3];
    int bc_lo[3], bc_hi[3];
    int sms;             // multiprocessors of the device (persistent grids are sized from it)
};

// non-uniform Cartesian spacing (Listing 1): per direction a device table [NU_NC][nus[d]] of the per-index
// WENO5 coefficients (beta_coef, poly_coef, d_cb of Listing 1) and the inverse cell width.  Only the table-driven
// instantiations (template flag NU) take this struct; the uniform ones take a plain Geo, so that their parameters and
// code are untouched by the feature.
struct GeoNu : Geo {
    const double *nu[3];
    int nus[3];          // row stride of nu[d] (p[d] plus padding, so that ragged tiles read defined entries)
};
template <bool NU> struct GeoOf { typedef Geo type; };
template <> struct GeoOf<true> { typedef GeoNu type; };

constexpr int NU_NC = 28;    // 9 beta_coef + 6 poly_coef (left) + 6 poly_coef (right) + 3 + 3 ideal weights + 1 / width

// stiffened-gas tables, PAPER.md:54-58 (Eq. 1), alpha-weighted mixture (reading B2)
struct Eos {
    // as given / as the definition divides by: used by the cons->prim kernel, which evaluates the
    // definition term by term without contraction
    double gamma[MAX_NF], pi_inf[MAX_NF], gm1[MAX_NF];
    double ygm1[MAX_NF]; // div_seed(gm1[i]) (mfc_math.cuh), computed on the device by launch_eos_seed
    // Gamma = G_last + sum_{i<nf-1} alpha_i dG_i ;  Pi likewise  (alpha_nf = 1 - sum alpha_i)
    double G_last, P_last, dG[MAX_NF], dP[MAX_NF];
    double weno_eps4;    // 4 * eps : smoothness indicators are carried scaled by 4
    int kapila;          // 1: K div(u) source of PAPER.md Eq. 2 on the alpha row (two fluids); 0: Allaire, K = 0
};

// output stage of one evaluation of L (a4 + a5):
//   out[cell] = base + coef * L(q)[cell],  base = cb * qs[cell] + ca * qn[cell]
//               (nbase = 0: base = 0;  nbase = 1: cb * qs only;  nbase = 2: both)
// mfc_rhs: coef = 1, nbase = 0.  RK stage: coef = cb * dt, so that
//   out = ca * qn + cb * (qs + dt * L(qs)).
// out must not alias the array L is evaluated on (blocks read their neighbours' cells of it as halo); it may
// alias qn, whose cell is read by the thread that writes it.
struct SweepOut {
    double *out;
    const double *qs, *qn;
    double ca, cb, coef;
    int nbase;
};

cudaError_t launch_prim(int ndim, int nf, const Geo &g, const Eos &e, const double *q, double *w, cudaStream_t s);
// 3D kernel: AUTO = the kernel with specialised Z warps (mfc_fused_roles.cuh) where it applies (TMA layout
// conditions), else the one-loop kernel staged by TMA boxes where the layout allows them (even padded extent in
// x, 16-byte aligned base), else per-thread cp.async; the other values force one of the three (and fail where it does not apply)
enum { MFC_PATH_AUTO = 0, MFC_PATH_TMA = 1, MFC_PATH_LDGSTS = 2, MFC_PATH_ROLES = 3 };
// g.nu[0] != nullptr selects the table-driven (non-uniform) instantiations
cudaError_t launch_rhs(int ndim, int nf, int order, const GeoNu &g, const Eos &e, const double *q, const SweepOut &o, int segment,
                       int path, cudaStream_t s);
cudaError_t launch_ghost_fill(const Geo &g, int neq, double *q, cudaStream_t s);
cudaError_t launch_cfl(int ndim, int nf, const GeoNu &g, const Eos &e, const double *q, unsigned long long *min_bits,
                       cudaStream_t s);
cudaError_t launch_eos_seed(const double *gm1_dev, double *ygm1_dev, int n, cudaStream_t s);
cudaError_t launch_line(int ndim, int nf, int order, int dir, const Eos &e, int n, const double *w, double *vL, double *vR,
                        double *F, double *uf, const double *nu, int nus, cudaStream_t s);

// per-dimension implementations
#define MFC_DECL_DIM(D)                                                                                               \
    cudaError_t launch_prim_d##D(int nf, const Geo &g, const Eos &e, const double *q, double *w, cudaStream_t s);     \
    cudaError_t launch_rhs_d##D(int nf, int order, const GeoNu &g, const Eos &e, const double *q, const SweepOut &o, int segment,  \
                                int path, cudaStream_t s);                                                            \
    cudaError_t launch_cfl_d##D(int nf, const GeoNu &g, const Eos &e, const double *q, unsigned long long *min_bits,  \
                                cudaStream_t s);                                                                      \
    cudaError_t launch_line_d##D(int nf, int order, int dir, const Eos &e, int n, const double *w, double *vL, double *vR,       \
                                 double *F, double *uf, const double *nu, int nus, cudaStream_t s);
MFC_DECL_DIM(1)
MFC_DECL_DIM(2)
MFC_DECL_DIM(3)
#undef MFC_DECL_DIM

}  // namespace mfc
