// kernels_vof.cuh -- SURVEY.md sec. 8(f) NEXT-4: one step of the MTHINC volume-of-fluid method (sec. 3.1,
// eqs. 8-12; Appendix A), triply periodic, linear reconstruction T(x~) = n . x~ (the curvature tensor of
// A.3-A.5 set to zero), directional splitting x -> y -> z (Algorithm 2):
//
//   per sweep p (s = n, x, y):   reconstruct  H^ = 1/2 [1 + tanh(beta (n . x~ + d))]  in every interface cell of phi^s
//                                flux through every face = integral of the UPWIND cell's H^ over the part swept in dt
//                                phi^p = [phi^s - (F_+ - F_-) / dl] / [1 - dt/dl (u_+ - u_-)]                       eq. (11)
//   finally                      phi^(n+1) = phi^z - sum_p dt/dl_p phi^p (u^p_+ - u^p_-)                             eq. (12)
//
//   n = m~ / |m~| with m~ the Youngs gradient in cell units (A.6): evaluated with explicitly rounded adds / multiplies in a
//       fixed order, because n decides an INTEGER -- the direction of exact integration, argmax |n| (cases 1-3,
//       PAPER.md:503-520) -- and that decision must not depend on fused multiply-adds;
//   d  from the volume constraint A.8 / A.10 in the paper's polynomial form (A.14-A.16): with D = e^{2 beta d},
//       A = e^{2 beta n_dir}, B_i = e^{2 beta a_i} (a_i = the transverse part of n . x~ at the four Gauss points) and
//       Q = e^{8 beta n_dir phi}:   prod_i (A B_i D + 1) = Q prod_i (B_i D + 1),  a quartic in D with exactly one positive
//       root, found by a bracketed Newton iteration on the polynomial, started from the root of the untilted case (robust
//       for every phi in (eps, 1 - eps), no transcendental function inside the iteration; the closed-form route A.17-A.21
//       is not used);
//   fluxes: exact integration of tanh along the sweep direction, 2 x 2 Gauss points across it (A.23-A.31).
//
// vof_flux_kernel<DIR>: a cell writes the flux of the faces it is the donor of (its + face when the velocity there is >= 0,
// its - face when the velocity there is < 0): every face is written exactly once.  The cells that carry a reconstruction
// are compacted per block before they are worked on (see the kernel).
// vof_update_kernel<DIR>: eq. (11).  vof_final_kernel: eq. (12).
#pragma once
#include "kernels.cuh"
#include "kernels_tma.cuh"   // rcp_normal

namespace flutas {

constexpr double kVofEps = 1e-8;
constexpr double kGauss0 = 0.5 - 0.28867513459481288225457439025098, kGauss1 = 0.5 + 0.28867513459481288225457439025098;

// Everything transcendental in a cell is an exponential of 2 beta n_c x~_c at a Gauss point or a cell face, so the
// reconstruction keeps the six numbers E[c][g] = e^{2 beta n_c g_g} (c = x, y, z; g_0, g_1 the Gauss points) and
// D = e^{2 beta d} instead of d itself:
//   * e^{2 beta (n . x~ + d)} at a Gauss point across a direction is a product of two E's and D;
//   * the volume constraint (A.14-A.16) is a polynomial in D whose coefficients are such products;
//   * with T(x) = e^{2 beta (alpha x + gamma)}:  int_a^b 1/2 [1 + tanh(beta (alpha x + gamma))] dx = ln[(1 + T(b)) / (1 + T(a))] / (2 beta alpha)
//     (ln cosh z = ln(e^{2z} + 1) - z - ln 2), so the mean over the four Gauss points across the sweep is ONE logarithm, of
//     the product of the four ratios, and T(a), T(b) are E_a G_i D, E_b G_i D with one new exponential per face.
// Per reconstructed cell and sweep: 8 exponentials and 1 logarithm (the first form of this kernel: 15 and 5).
struct VofRecon {
    double n[3];
    double E[3][2];      // e^{2 beta n_c g0}, e^{2 beta n_c g1}
    double D;            // e^{2 beta d}
    bool flat;           // no reconstruction: the cell carries the constant state phi
};

// reconstruction of cell (i, j, k), phi(i, j, k) = fc in (eps, 1 - eps), from the field f (periodic)
__device__ __forceinline__ void vof_reconstruct(const GridParams &g, const double *__restrict__ f, int i, int j, int k, double fc,
                                                double beta, VofRecon &r) {
    const long long sy = g.nx, sz = (long long)g.nx * g.ny;
    r.flat = true; r.D = 1.0; r.n[0] = r.n[1] = r.n[2] = 0.0;
    int ii[3] = {i == 0 ? g.nx - 1 : i - 1, i, i == g.nx - 1 ? 0 : i + 1};
    int jj[3] = {j == 0 ? g.ny - 1 : j - 1, j, j == g.ny - 1 ? 0 : j + 1};
    int kk[3] = {k == 0 ? g.nz - 1 : k - 1, k, k == g.nz - 1 ? 0 : k + 1};
    double p[3][3][3];   // [dk][dj][di]
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) p[c][b][a] = __ldg(f + ii[a] + sy * jj[b] + sz * kk[c]);
    // Youngs: the gradient at the 8 corners from the 8 cells around each, then their mean.  Explicitly rounded operations
    // in a fixed order (corner order k, j, i): no fused multiply-add may change n, which decides the integration direction.
    double m0 = 0.0, m1 = 0.0, m2 = 0.0;
#pragma unroll
    for (int ck = 0; ck < 2; ++ck)
#pragma unroll
        for (int cj = 0; cj < 2; ++cj)
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const double p000 = p[ck][cj][ci], p100 = p[ck][cj][ci + 1], p010 = p[ck][cj + 1][ci], p110 = p[ck][cj + 1][ci + 1];
                const double p001 = p[ck + 1][cj][ci], p101 = p[ck + 1][cj][ci + 1], p011 = p[ck + 1][cj + 1][ci], p111 = p[ck + 1][cj + 1][ci + 1];
                auto sum4 = [](double a, double b, double c, double d) { return __dadd_rn(__dadd_rn(__dadd_rn(a, b), c), d); };
                m0 = __dadd_rn(m0, __dmul_rn(0.25, sum4(__dsub_rn(p100, p000), __dsub_rn(p110, p010), __dsub_rn(p101, p001), __dsub_rn(p111, p011))));
                m1 = __dadd_rn(m1, __dmul_rn(0.25, sum4(__dsub_rn(p010, p000), __dsub_rn(p110, p100), __dsub_rn(p011, p001), __dsub_rn(p111, p101))));
                m2 = __dadd_rn(m2, __dmul_rn(0.25, sum4(__dsub_rn(p001, p000), __dsub_rn(p101, p100), __dsub_rn(p011, p010), __dsub_rn(p111, p110))));
            }
    m0 = __dmul_rn(m0, 0.125); m1 = __dmul_rn(m1, 0.125); m2 = __dmul_rn(m2, 0.125);
    const double mag = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(m0, m0), __dmul_rn(m1, m1)), __dmul_rn(m2, m2)));
    if (!(mag > 1e-12)) return;
    r.flat = false;
    r.n[0] = m0 / mag; r.n[1] = m1 / mag; r.n[2] = m2 / mag;
    const double tb = 2.0 * beta;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        r.E[c][0] = exp(tb * r.n[c] * kGauss0);
        r.E[c][1] = exp(tb * r.n[c] * kGauss1);
    }
    const double ax = fabs(r.n[0]), ay = fabs(r.n[1]), az = fabs(r.n[2]);
    const int dir = (ax >= ay && ax >= az) ? 0 : ((ay >= az) ? 1 : 2);     // direction of exact integration (cases 1-3)
    double nd = dir == 0 ? r.n[0] : (dir == 1 ? r.n[1] : r.n[2]);
    double A = dir == 0 ? r.E[0][0] * r.E[0][1] : (dir == 1 ? r.E[1][0] * r.E[1][1] : r.E[2][0] * r.E[2][1]);   // e^{2 beta n_dir}
    double P0 = dir == 0 ? r.E[1][0] : (dir == 1 ? r.E[2][0] : r.E[0][0]), P1 = dir == 0 ? r.E[1][1] : (dir == 1 ? r.E[2][1] : r.E[0][1]);
    double R0 = dir == 0 ? r.E[2][0] : (dir == 1 ? r.E[0][0] : r.E[1][0]), R1 = dir == 0 ? r.E[2][1] : (dir == 1 ? r.E[0][1] : r.E[1][1]);
    double qq = exp(tb * nd * fc);
    // Cells more than half full are solved as their mirror image (n -> -n, phi -> 1 - phi, D -> 1 / D: the same polynomial with
    // every coefficient replaced by its reciprocal and Q by Q / A^4): the iteration below converges in 4-5 steps from the
    // dilute side and needs about twice as many from the other.
    const bool mirror = fc > 0.5;
    if (mirror) {
        A = rcp_normal(A); P0 = rcp_normal(P0); P1 = rcp_normal(P1); R0 = rcp_normal(R0); R1 = rcp_normal(R1);
        qq *= A; nd = -nd;
    }
    // prod_i (A B_i D + 1) = Q prod_i (B_i D + 1)   (A.14-A.16 with Q here = A^2 Q_paper), B_i = e^{2 beta a_i}
    const double B0 = P0 * R0, B1 = P0 * R1, B2 = P1 * R0, B3 = P1 * R1;
    const double AB0 = A * B0, AB1 = A * B1, AB2 = A * B2, AB3 = A * B3;
    const double q2 = qq * qq, Q = q2 * q2;
    // F(D) = sgn [ prod (A B_i D + 1) - Q prod (B_i D + 1) ], sgn = sign(n_dir): increasing in D, F(0) < 0 < F(inf), exactly one
    // positive root (ln of the ratio of the two products rises monotonically from 0 to 4 ln A).  Newton's iteration on the
    // polynomial and its derivative (product rule, no division), kept inside a bracket (a step that would leave it is replaced
    // by a bisection).  With no transverse tilt (B_i = 1) the root is c = (q - 1) / (A - q), q = Q^(1/4).  One reciprocal
    // (hardware seed + two Newton steps on it) and about 35 multiply-adds per iteration, 4-6 iterations on average, no
    // transcendental function.
    // The root is bracketed rigorously: every factor (A B_i D + 1) / (B_i D + 1) is monotone in B_i D, so with all B_i replaced
    // by the largest (smallest) one the root is c / B_max (c / B_min); the geometric mean of the B_i gives the starting point.
    const double sgn = nd > 0.0 ? 1.0 : -1.0;
    // (reciprocals by rcp_normal: <= ~1 ulp, the bracket is widened by far more than that)
    const double c0 = (qq - 1.0) * rcp_normal(A - qq);
    const double bmin = fmin(fmin(B0, B1), fmin(B2, B3)), bmax = fmax(fmax(B0, B1), fmax(B2, B3));
    double lo = c0 * rcp_normal(bmax) * (1.0 - 1.0e-14), hi = c0 * rcp_normal(bmin) * (1.0 + 1.0e-14), x = c0 * rsqrt(B0 * B3), prev_step = 1.0e300;
    for (int it = 0; it < 64; ++it) {
        const double f0 = fma(AB0, x, 1.0), f1 = fma(AB1, x, 1.0), f2 = fma(AB2, x, 1.0), f3 = fma(AB3, x, 1.0);
        const double g0 = fma(B0, x, 1.0), g1 = fma(B1, x, 1.0), g2 = fma(B2, x, 1.0), g3 = fma(B3, x, 1.0);
        const double n01 = f0 * f1, n23 = f2 * f3, m01 = g0 * g1, m23 = g2 * g3;
        const double Fv = sgn * fma(-Q, m01 * m23, n01 * n23);
        const double dN = fma(fma(AB0, f1, AB1 * f0), n23, n01 * fma(AB2, f3, AB3 * f2));
        const double dM = fma(fma(B0, g1, B1 * g0), m23, m01 * fma(B2, g3, B3 * g2));
        const double dF = sgn * fma(-Q, dM, dN);
        if (fabs(Fv) <= 2.0e-15 * (n01 * n23)) break;        // the two products agree to round-off: nothing left to gain
        if (Fv < 0.0) lo = x; else hi = x;
        double xn = dF > 0.0 ? fma(-Fv, rcp_normal(dF), x) : -1.0;
        if (dF > 0.0 && fabs(xn - x) <= 4.0e-16 * x) { x = xn; break; }          // the step is below the resolution of x
        const bool fallback = !(xn > lo) || !(xn < hi);                          // left the bracket (or no usable derivative)
        if (fallback) xn = Fv < 0.0 ? 0.5 * (x + hi) : 0.5 * (lo + x);
        const double step = fabs(xn - x);
        x = xn;
        if (step <= 4.0e-16 * x) break;
        // Newton's steps shrink faster than geometrically until they reach round-off level: the first one that does not is noise
        if (!fallback && step <= 1.0e-3 * x && step >= 0.5 * prev_step) break;
        prev_step = fallback ? 1.0e300 : step;
    }
    const double root = mirror ? rcp_normal(x) : x;
    r.D = root;
}

// mean of H^ over x~_DIR in [a, b] x the unit square across DIR, times (b - a) -- i.e. the volume of fluid in that slice
template <int DIR>
__device__ __forceinline__ double vof_slice(const VofRecon &r, double a, double b, double beta) {
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    const double alpha = r.n[DIR], tb = 2.0 * beta;
    // e^{2 beta gamma_i} at the four Gauss points across DIR
    const double G0 = r.E[T1][0] * r.E[T2][0] * r.D, G1 = r.E[T1][0] * r.E[T2][1] * r.D;
    const double G2 = r.E[T1][1] * r.E[T2][0] * r.D, G3 = r.E[T1][1] * r.E[T2][1] * r.D;
    if (fabs(alpha) < 1e-12)      // 1/2 (1 + tanh z) = e^{2z} / (1 + e^{2z})
        return (b - a) * 0.25 * (G0 * rcp_normal(1.0 + G0) + G1 * rcp_normal(1.0 + G1) + G2 * rcp_normal(1.0 + G2) + G3 * rcp_normal(1.0 + G3));
    // mean over the four Gauss points of int_a^b = ln[ prod_i (1 + E_b G_i) / prod_i (1 + E_a G_i) ] / (4 * 2 beta alpha), E_x = e^{2 beta alpha x}.
    // The quotient is 1 + O(2 beta alpha (b - a)): for a normal almost perpendicular to the sweep, or a thin slice, its
    // logarithm would lose the leading digits of that increment (|alpha| = 1e-9 leaves 7).  So the quotient is never formed:
    // with "lo" the end of [a, b] with the smaller exponent and e = e^{|2 beta alpha (b - a)|} - 1 >= 0, every factor at the
    // other end is the factor at lo plus e h_i (h_i = E_lo G_i), the difference of the two products is e times a polynomial
    // in e with positive coefficients -- no subtraction anywhere -- and the result is +- log1p(e poly / prod_lo), accurate for
    // every alpha.  One expm1 and one log1p per face (before: one exp and one log); E_lo follows from the known end
    // (E_0 = 1, E_1 = the cell's table) without another exponential.
    const double dl = tb * alpha * (b - a);
    const bool up = dl >= 0.0;                                   // lo = a (up) or b
    const double e = expm1(fabs(dl)), E1 = r.E[DIR][0] * r.E[DIR][1];
    const double Elo = up ? (a == 0.0 ? 1.0 : (b == 1.0 ? E1 * rcp_normal(1.0 + e) : exp(tb * alpha * a)))
                          : (b == 1.0 ? E1 : (a == 0.0 ? rcp_normal(1.0 + e) : exp(tb * alpha * b)));
    const double h0 = Elo * G0, h1 = Elo * G1, h2 = Elo * G2, h3 = Elo * G3;
    const double d0 = 1.0 + h0, d1 = 1.0 + h1, d2 = 1.0 + h2, d3 = 1.0 + h3;
    const double A0 = d0 * d1, A1 = fma(d0, h1, h0 * d1), A2 = h0 * h1;      // (d0 + e h0)(d1 + e h1) = A0 + e A1 + e^2 A2
    const double B0 = d2 * d3, B1 = fma(d2, h3, h2 * d3), B2 = h2 * h3;
    const double c1 = fma(A0, B1, A1 * B0), c2 = fma(A0, B2, fma(A1, B1, A2 * B0)), c3 = fma(A1, B2, A2 * B1), c4 = A2 * B2;
    const double x = e * fma(e, fma(e, fma(e, c4, c3), c2), c1) * rcp_normal(A0 * B0);
    const double L = log1p(x);
    return (up ? L : -L) * rcp_normal(4.0 * tb * alpha);
}

// A block owns VofTile::CELLS consecutive cells.  Pass 1: every cell finds out which of its faces it is the donor of (its +
// face when the velocity there is >= 0, its - face when the velocity there is < 0: every face is written exactly once) and
// either writes the flux of a constant state at once or -- phi in (eps, 1 - eps) -- joins the block's work list.  Pass 2:
// the list is worked off with every lane busy (the cells that carry a reconstruction are a band around the interfaces:
// one cell in a warp of consecutive cells here, ten there).
struct VofTile { static constexpr int NT = 256, PER = 4, CELLS = NT * PER; };

template <int DIR>
__global__ void __launch_bounds__(VofTile::NT, 4)
vof_flux_kernel(GridParams g, double beta, double dt, const double *__restrict__ phi, const double *__restrict__ vel,
                double *__restrict__ flux) {
    using T = VofTile;
    __shared__ int list[T::CELLS];
    __shared__ int n_list;
    const long long npts = (long long)g.nx * g.ny * g.nz, base = (long long)blockIdx.x * T::CELLS;
    const long long sy = g.nx, sz = (long long)g.nx * g.ny;
    const double dl = 1.0 / (DIR == 0 ? g.inv_dx : (DIR == 1 ? g.inv_dy : g.inv_dz));
    const double dt_dl = dt / dl;
    auto minus_of = [&](long long q, int i, int j, int k) {
        return DIR == 0 ? (i == 0 ? q + (g.nx - 1) : q - 1) : DIR == 1 ? (j == 0 ? q + (g.ny - 1) * sy : q - sy) : (k == 0 ? q + (g.nz - 1) * sz : q - sz);
    };
    if (threadIdx.x == 0) n_list = 0;
    __syncthreads();
#pragma unroll
    for (int c = 0; c < T::PER; ++c) {
        const int loc = c * T::NT + threadIdx.x;
        const long long q = base + loc;
        bool queued = false;
        if (q < npts) {
            const int i = (int)(q % g.nx), j = (int)((q / g.nx) % g.ny), k = (int)(q / sz);
            const long long qm = minus_of(q, i, j, k);
            const double cp = vel[q] * dt_dl, cm = vel[qm] * dt_dl;              // local CFL numbers on the + and - face (A.26)
            const bool give_p = cp >= 0.0, give_m = cm < 0.0;
            if (give_p || give_m) {
                const double fc = phi[q];
                if (fc > kVofEps && fc < 1.0 - kVofEps) queued = true;
                else {
                    if (give_p) flux[q] = dl * (cp * fc);
                    if (give_m) flux[qm] = -dl * (-cm * fc);
                }
            }
        }
        // warp-aggregated append
        const unsigned m = __ballot_sync(0xffffffffu, queued);
        int pos = 0;
        if ((threadIdx.x & 31) == 0 && m) pos = atomicAdd(&n_list, __popc(m));
        pos = __shfl_sync(0xffffffffu, pos, 0);
        if (queued) list[pos + __popc(m & ((1u << (threadIdx.x & 31)) - 1u))] = loc;
    }
    __syncthreads();
    const int n = n_list;
    for (int it = threadIdx.x; it < n; it += T::NT) {
        const long long q = base + list[it];
        const int i = (int)(q % g.nx), j = (int)((q / g.nx) % g.ny), k = (int)(q / sz);
        const long long qm = minus_of(q, i, j, k);
        const double cp = vel[q] * dt_dl, cm = vel[qm] * dt_dl;
        const bool give_p = cp >= 0.0, give_m = cm < 0.0;
        const double fc = phi[q];
        VofRecon r;
        vof_reconstruct(g, phi, i, j, k, fc, beta, r);
        if (give_p)                                                              // the last cp of the way through this cell
            flux[q] = dl * (r.flat ? cp * fc : vof_slice<DIR>(r, 1.0 - cp, 1.0, beta));
        if (give_m)                                                              // the first |cm| of it, leaving backwards
            flux[qm] = -dl * (r.flat ? -cm * fc : vof_slice<DIR>(r, 0.0, -cm, beta));
    }
}

template <int DIR>
__global__ void __launch_bounds__(256)
vof_update_kernel(GridParams g, double dt, const double *__restrict__ phi, const double *__restrict__ vel,
                  const double *__restrict__ flux, double *__restrict__ out) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long npts = (long long)g.nx * g.ny * g.nz;
    if (q >= npts) return;
    const int i = (int)(q % g.nx), j = (int)((q / g.nx) % g.ny), k = (int)(q / ((long long)g.nx * g.ny));
    const long long sy = g.nx, sz = (long long)g.nx * g.ny;
    const long long qm = DIR == 0 ? (i == 0 ? q + (g.nx - 1) : q - 1)
                       : DIR == 1 ? (j == 0 ? q + (g.ny - 1) * sy : q - sy) : (k == 0 ? q + (g.nz - 1) * sz : q - sz);
    const double inv_dl = DIR == 0 ? g.inv_dx : (DIR == 1 ? g.inv_dy : g.inv_dz);
    const double du = vel[q] - vel[qm];
    out[q] = (phi[q] - (flux[q] - flux[qm]) * inv_dl) / (1.0 - dt * inv_dl * du);     // eq. (11)
}

__global__ void __launch_bounds__(256)
vof_final_kernel(GridParams g, double dt, const double *__restrict__ px, const double *__restrict__ py, const double *__restrict__ pz,
                 const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w, double *__restrict__ out) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long npts = (long long)g.nx * g.ny * g.nz;
    if (q >= npts) return;
    const int i = (int)(q % g.nx), j = (int)((q / g.nx) % g.ny), k = (int)(q / ((long long)g.nx * g.ny));
    const long long sy = g.nx, sz = (long long)g.nx * g.ny;
    const double du = u[q] - u[i == 0 ? q + (g.nx - 1) : q - 1];
    const double dv = v[q] - v[j == 0 ? q + (g.ny - 1) * sy : q - sy];
    const double dw = w[q] - w[k == 0 ? q + (g.nz - 1) * sz : q - sz];
    out[q] = pz[q] - (dt * g.inv_dx * px[q] * du + dt * g.inv_dy * py[q] * dv + dt * g.inv_dz * pz[q] * dw);   // eq. (12)
}

}  // namespace flutas
