/*
 * oscnet_oracle.c  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU restatement of the hot path of
 * arXiv:2410.19075 (Sudakov & Maistrenko): fixed-step classical RK4 of N
 * coupled oscillators whose right-hand side is "local vector field + sum over
 * the in-neighbours the topology allows".  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this file.  It
 * shares no code, header, table or constant generator with the CUDA library
 * under paper_2410_19075_b200/csrc/.
 *
 * Decomposition = the paper's: parallel over elements, each element's neighbour
 * sum serial, in ascending neighbour index ("The right-hand part
 * of the differential equation for each individual oscillator is computed
 * serially as described by Algorithm 1"; Alg. 1).
 * No algebraic rewrites (no factorised sine, no prefix sums, no tiling) -- with one
 * fenced exception at the end of the file (ora_rhs_fast / ora_rk4_fast), which SURVEY.md
 * 8(c) allows for the long statistics runs only and which is pinned against ora_rhs.
 *
 * Readings of the paper that this file takes are the DESIGN.md "Readings"
 * table (R1..R14); each function names the ones it uses.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   ora_topology_ring / _lattice : ball sizes 33 (P=2) and 925 (P=6) printed in
 *       PAPER.md:337-339 (tests/golden/lattice_link_counts.txt), symmetry,
 *       dense-matrix brute force, index map k*N1^2+j*N1+i.
 *   ora_topology_random_indegree : exactly k distinct sources != i, sorted;
 *       re-derived in pure Python integers on tiny cases.
 *   ora_rhs (KS)  : K=0 closed form, in-phase invariance, sum conservation for
 *       alpha=0, mean-field identity on all-to-all rings, dense brute force.
 *   ora_rhs (FHN) : closed-form fixed point (-a, -a+a^3/3), vanishing coupling
 *       on uniform states, zero-sum coupling, dense brute force.
 *   ora_rhs (HH)  : hand-computed rate values at V=-65 mV, rest state near the
 *       textbook -65 mV / m=0.0529 h=0.5961 n=0.3177, dense brute force.
 *   ora_rhs (KSI) : (Kuramoto-Sakaguchi with inertia) dense
 *       brute force, in-phase state, momentum balance for alpha=0, damped closed form for K=0.
 *   ora_rk4       : 4th-order convergence against a 16x finer step; exactness
 *       for constant RHS.
 *   ora_local_order, phase maps : R=1 for identical phases, splay state R=0.
 *   Long-run order-parameter statistics of the coupled configs: PARITY UNPINNED in absolute
 *       terms (the paper prints no value); they are only compared GPU-vs-oracle.  The procedure
 *       (oracle.py: run_statistics) is pinned on the K = 0 closed form.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORA_MODEL_KS 0
#define ORA_MODEL_FHN 1
#define ORA_MODEL_HH 2
#define ORA_MODEL_KSI 3   /* Kuramoto-Sakaguchi with inertia, eq. (3) in full (next row) */
#define ORA_MODEL_FHN2 4  /* FitzHugh-Nagumo exactly as eq. (2): x-only coupling, delay, noise, I_app (8(f).4) */
#define ORA_MODEL_HHS 5   /* Hodgkin-Huxley with the synaptic gating ODE of eq. (1) (8(f).4) */

/* ------------------------------------------------------------------ */
/* Topology: canonical CSR, rows = in-neighbour lists (PAPER.md:147:    */
/* L_ij = 1 iff j influences i), sorted ascending, int64 row_ptr,       */
/* int32 col_idx.  Row ranges [row_begin, row_begin+row_count) so that  */
/* huge lattices can be sampled; row_ptr is relative to the range.      */
/* ------------------------------------------------------------------ */

static int cmp_i32(const void* a, const void* b) {
    int32_t x = *(const int32_t*)a, y = *(const int32_t*)b;
    return (x > y) - (x < y);
}

/* 1D ring: "each oscillator is coupled with its P neighbors on both sides" on
 * a circle.  j = (i + d) mod n, d in [-P, P], d != 0 unless
 * include_self (reading R4). */
int ora_topology_ring(int64_t n, int32_t P, int32_t include_self, int64_t row_begin,
                      int64_t row_count, int64_t* row_ptr, int32_t* col_idx) {
    if (n < 1 || P < 0 || 2 * (int64_t)P >= n) return -1;
    int64_t pos = 0;
    for (int64_t r = 0; r < row_count; ++r) {
        int64_t i = row_begin + r;
        row_ptr[r] = pos;
        int64_t start = pos;
        for (int64_t d = -P; d <= P; ++d) {
            if (d == 0 && !include_self) continue;
            int64_t j = (i + d) % n;
            if (j < 0) j += n;
            col_idx[pos++] = (int32_t)j;
        }
        qsort(col_idx + start, (size_t)(pos - start), sizeof(int32_t), cmp_i32);
    }
    row_ptr[row_count] = pos;
    return 0;
}

/* Number of lattice points d with |d|^2 <= P^2 (minus the centre unless
 * include_self).  PAPER.md:309 (2D disc), :313 (3D ball). */
int64_t ora_lattice_degree(int32_t ndim, int32_t P, int32_t include_self) {
    int64_t c = 0;
    int32_t Pz = ndim >= 3 ? P : 0, Py = ndim >= 2 ? P : 0;
    for (int32_t dz = -Pz; dz <= Pz; ++dz)
        for (int32_t dy = -Py; dy <= Py; ++dy)
            for (int32_t dx = -P; dx <= P; ++dx)
                if (dx * dx + dy * dy + dz * dz <= P * P) ++c;
    return include_self ? c : c - 1;
}

/* d-dimensional periodic lattice.  Site (i,j,k) <-> index k*nx*ny + j*nx + i
 * (PAPER.md:309 "jN1+i", :311 "kN1^2+jN1+i"); neighbours = all sites with
 * (i-i')^2+(j-j')^2+(k-k')^2 <= P^2, coordinates taken modulo
 * the extent ("torus"). */
int ora_topology_lattice(int32_t ndim, const int64_t* extent, int32_t P, int32_t include_self,
                         int64_t row_begin, int64_t row_count, int64_t* row_ptr,
                         int32_t* col_idx) {
    if (ndim < 1 || ndim > 3 || P < 0) return -1;
    int64_t nx = extent[0], ny = ndim >= 2 ? extent[1] : 1, nz = ndim >= 3 ? extent[2] : 1;
    if (2 * (int64_t)P >= nx) return -1;
    if (ndim >= 2 && 2 * (int64_t)P >= ny) return -1;
    if (ndim >= 3 && 2 * (int64_t)P >= nz) return -1;
    int32_t Pz = ndim >= 3 ? P : 0, Py = ndim >= 2 ? P : 0;
    int64_t pos = 0;
    for (int64_t r = 0; r < row_count; ++r) {
        int64_t idx = row_begin + r;
        int64_t i = idx % nx, j = (idx / nx) % ny, k = idx / (nx * ny);
        row_ptr[r] = pos;
        int64_t start = pos;
        for (int32_t dz = -Pz; dz <= Pz; ++dz)
            for (int32_t dy = -Py; dy <= Py; ++dy)
                for (int32_t dx = -P; dx <= P; ++dx) {
                    if (dx * dx + dy * dy + dz * dz > P * P) continue;
                    if (dx == 0 && dy == 0 && dz == 0 && !include_self) continue;
                    int64_t ii = ((i + dx) % nx + nx) % nx;
                    int64_t jj = ((j + dy) % ny + ny) % ny;
                    int64_t kk = ((k + dz) % nz + nz) % nz;
                    col_idx[pos++] = (int32_t)(kk * nx * ny + jj * nx + ii);
                }
        qsort(col_idx + start, (size_t)(pos - start), sizeof(int32_t), cmp_i32);
    }
    row_ptr[row_count] = pos;
    return 0;
}

/* Reading R8: seeded random graph with fixed in-degree k, uniform sources, no
 * self-loops, no multi-edges.  Integer-only and counter-based so that any
 * other implementation of the same rule is bit-exact:
 *   mix(z): z ^= z>>30; z *= 0xBF58476D1CE4E5B9; z ^= z>>27;
 *           z *= 0x94D049BB133111EB; z ^= z>>31        (splitmix64 finaliser)
 *   h(seed,i,t) = mix( mix(seed + G*(i+1)) + G*(t+1) ),  G = 0x9E3779B97F4A7C15
 *   candidate  j = floor(h * (n-1) / 2^64);  if j >= i then j += 1
 * for t = 0,1,2,...; a candidate already in the row is skipped; the row is the
 * first k distinct candidates, sorted ascending. */
uint64_t ora_mix64(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

int ora_topology_random_indegree(int64_t n, int32_t k, uint64_t seed, int64_t row_begin,
                                 int64_t row_count, int64_t* row_ptr, int32_t* col_idx) {
    if (n < 2 || k < 0 || (int64_t)k > n - 1) return -1;
    const uint64_t G = 0x9E3779B97F4A7C15ULL;
    for (int64_t r = 0; r < row_count; ++r) {
        int64_t i = row_begin + r;
        int32_t* row = col_idx + r * (int64_t)k;
        row_ptr[r] = r * (int64_t)k;
        uint64_t hi = ora_mix64(seed + G * (uint64_t)(i + 1));
        int32_t have = 0;
        for (uint64_t t = 0; have < k; ++t) {
            uint64_t h = ora_mix64(hi + G * (t + 1));
            uint64_t j = (uint64_t)(((unsigned __int128)h * (unsigned __int128)(uint64_t)(n - 1)) >> 64);
            if (j >= (uint64_t)i) j += 1;
            int dup = 0;
            for (int32_t q = 0; q < have; ++q)
                if (row[q] == (int32_t)j) { dup = 1; break; }
            if (!dup) row[have++] = (int32_t)j;
        }
        qsort(row, (size_t)k, sizeof(int32_t), cmp_i32);
    }
    row_ptr[row_count] = row_count * (int64_t)k;
    return 0;
}

/* ------------------------------------------------------------------ */
/* Network description handed to the RHS / integrator.                  */
/* State is SoA: y[var*n + i].                                           */
/*   KS : var 0 = phi                          elem_param = omega[n]     */
/*   FHN: var 0 = u, 1 = v                     elem_param unused         */
/*   HH : var 0 = V, 1 = m, 2 = h, 3 = n       elem_param = I_ext[n]     */
/* p[] per model:                                                        */
/*   KS : K, alpha                                                       */
/*   FHN: eps, a, sigma, b_uu, b_uv, b_vu, b_vv                          */
/*   HH : gNa, gK, gL, ENa, EK, EL, C, g_syn, E_syn, theta_syn, k_syn    */
/* ------------------------------------------------------------------ */
typedef struct {
    int32_t model;
    int32_t pad_;
    int64_t n;
    const int64_t* row_ptr; /* n+1 */
    const int32_t* col_idx;
    const double* elem_param;
    double p[16];
} ora_net;

int32_t ora_nvar(int32_t model) {
    return model == ORA_MODEL_KS ? 1 : model == ORA_MODEL_FHN ? 2 : model == ORA_MODEL_HH ? 4 :
           model == ORA_MODEL_KSI ? 2 : model == ORA_MODEL_FHN2 ? 2 : model == ORA_MODEL_HHS ? 5 : -1;
}

/* Kuramoto-Sakaguchi (eq. (3) with m=0, eps=1, mu=1/Omega, PAPER.md:79, :107;
 * Alg. 1) with natural frequency and strength K as the
 * north-star configs state them:
 *   f_i = omega_i + (K/Omega_i) * sum_{j in row i} sin(phi_j - phi_i - alpha)
 * Omega_i = number of links actually iterated; the division happens once,
 * after the loop (reading R2 of the garbled listing). */
static void rhs_ks(const ora_net* net, const double* y, double* f) {
    const int64_t n = net->n;
    const double K = net->p[0], alpha = net->p[1];
    const double* phi = y;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double der = 0.0;
        int64_t links_amount = 0;
        for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e, ++links_amount) {
            int32_t j = net->col_idx[e];
            der += sin(phi[j] - phi[i] - alpha);
        }
        if (links_amount > 0) der /= (double)links_amount;
        f[i] = net->elem_param[i] + K * der;
    }
}

/* Kuramoto-Sakaguchi with inertia, eq. (3) PAPER.md:79 in full:
 *   m phi_i'' + eps phi_i' = mu sum_j L_ij sin(phi_j - phi_i - alpha),
 * the model of the paper's own performance tests (Fig. 6c: m = 1,
 * eps = 0.05, mu = 0.01, 3D ball of radius 2 / 4 / 6).  As a first-order system in (phi, psi = phi'):
 *   phi_i' = psi_i
 *   psi_i' = ( -eps psi_i + omega_i + (K/Omega_i) sum_{j in row i} sin(phi_j - phi_i - alpha) ) / m
 * with the coupling normalised as in rhs_ks (K/Omega_i = mu; reading R2) and an optional constant
 * torque omega_i (0 in the paper).  State SoA [phi | psi].  p = {K, alpha, m, eps}.
 * Pins (tests/test_oracle_dynamics.py): dense brute force, in-phase state, momentum balance
 * sum_i psi_i' = -(eps/m) sum_i psi_i + sum_i omega_i / m for alpha = 0 on symmetric topologies, the
 * damped closed form for K = 0 within the RK4 truncation error, reduction to rhs_ks as m -> 0 is
 * NOT used (singular limit). */
static void rhs_ksi(const ora_net* net, const double* y, double* f) {
    const int64_t n = net->n;
    const double K = net->p[0], alpha = net->p[1], m = net->p[2], eps = net->p[3];
    const double* phi = y;
    const double* psi = y + n;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double der = 0.0;
        int64_t links_amount = 0;
        for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e, ++links_amount) {
            int32_t j = net->col_idx[e];
            der += sin(phi[j] - phi[i] - alpha);
        }
        if (links_amount > 0) der /= (double)links_amount;
        f[i] = psi[i];
        f[n + i] = (-eps * psi[i] + net->elem_param[i] + K * der) / m;
    }
}

/* FitzHugh-Nagumo, eq. (2) PAPER.md:70-75 in the north-star variant (reading
 * R3): rotated 2x2 diffusive coupling on (u,v), no delay, no noise, no I_app.
 *   Cu_i = sum_j (u_j - u_i),  Cv_i = sum_j (v_j - v_i)   over row i
 *   eps du_i/dt = u_i - u_i^3/3 - v_i + (sigma/Omega_i)(b_uu Cu_i + b_uv Cv_i)
 *       dv_i/dt = u_i + a            + (sigma/Omega_i)(b_vu Cu_i + b_vv Cv_i) */
static void rhs_fhn(const ora_net* net, const double* y, double* f) {
    const int64_t n = net->n;
    const double eps = net->p[0], a = net->p[1], sigma = net->p[2];
    const double buu = net->p[3], buv = net->p[4], bvu = net->p[5], bvv = net->p[6];
    const double* u = y;
    const double* v = y + n;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double Cu = 0.0, Cv = 0.0;
        int64_t links_amount = 0;
        for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e, ++links_amount) {
            int32_t j = net->col_idx[e];
            Cu += u[j] - u[i];
            Cv += v[j] - v[i];
        }
        double s = links_amount > 0 ? sigma / (double)links_amount : 0.0;
        f[i] = (u[i] - u[i] * u[i] * u[i] / 3.0 - v[i] + s * (buu * Cu + buv * Cv)) / eps;
        f[n + i] = u[i] + a + s * (bvu * Cu + bvv * Cv);
    }
}

/* x / (1 - exp(-x/10)) with its removable singularity at x = 0 (reading R10):
 * -x/expm1(-x/10), and the limit 10 when |x/10| < 1e-9. */
static double hh_vtrap(double x) {
    if (fabs(x / 10.0) < 1e-9) return 10.0;
    return -x / expm1(-x / 10.0);
}

/* Standard squid-axon rate functions, rest near -65 mV (reading R7; mV, ms). */
static void hh_rates(double V, double* am, double* bm, double* ah, double* bh, double* an,
                     double* bn) {
    *am = 0.1 * hh_vtrap(V + 40.0);
    *bm = 4.0 * exp(-(V + 65.0) / 18.0);
    *ah = 0.07 * exp(-(V + 65.0) / 20.0);
    *bh = 1.0 / (1.0 + exp(-(V + 35.0) / 10.0));
    *an = 0.01 * hh_vtrap(V + 55.0);
    *bn = 0.125 * exp(-(V + 65.0) / 80.0);
}

/* Hodgkin-Huxley type element, eq. (1), in the north-star
 * variant (reading R7): instantaneous sigmoidal synapse S(V_pre),
 *   C dV_i/dt = I_ext,i - gNa m^3 h (V-ENa) - gK n^4 (V-EK) - gL (V-EL)
 *               + (g_syn/Omega_i) (E_syn - V_i) sum_{j in row i} S(V_j)
 *   dx/dt = alpha_x(V)(1-x) - beta_x(V) x,  x in {m,h,n}
 *   S(V) = 1/(1+exp(-(V-theta_syn)/k_syn)). */
static void rhs_hh(const ora_net* net, const double* y, double* f) {
    const int64_t n = net->n;
    const double gNa = net->p[0], gK = net->p[1], gL = net->p[2];
    const double ENa = net->p[3], EK = net->p[4], EL = net->p[5], C = net->p[6];
    const double gsyn = net->p[7], Esyn = net->p[8], th = net->p[9], ks = net->p[10];
    const double *V = y, *m = y + n, *h = y + 2 * n, *g = y + 3 * n;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double ssum = 0.0;
        int64_t links_amount = 0;
        for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e, ++links_amount) {
            int32_t j = net->col_idx[e];
            ssum += 1.0 / (1.0 + exp(-(V[j] - th) / ks));
        }
        double Isyn = links_amount > 0 ? (gsyn / (double)links_amount) * (Esyn - V[i]) * ssum : 0.0;
        double am, bm, ah, bh, an, bn;
        hh_rates(V[i], &am, &bm, &ah, &bh, &an, &bn);
        double INa = gNa * m[i] * m[i] * m[i] * h[i] * (V[i] - ENa);
        double IK = gK * g[i] * g[i] * g[i] * g[i] * (V[i] - EK);
        double IL = gL * (V[i] - EL);
        f[i] = (net->elem_param[i] - INa - IK - IL + Isyn) / C;
        f[n + i] = am * (1.0 - m[i]) - bm * m[i];
        f[2 * n + i] = ah * (1.0 - h[i]) - bh * h[i];
        f[3 * n + i] = an * (1.0 - g[i]) - bn * g[i];
    }
}

/* FitzHugh-Nagumo exactly as the paper prints it, eq. (2) PAPER.md:70-75:
 *   eps dx_i/dt = x_i - x_i^3/3 - y_i + sum_j L_ij s_ij (x_j(t - tau) - x_i) + I_app
 *       dy_i/dt = x_i + a + D n(t)
 * with uniform coupling strength s_ij = sigma / Omega_i (reading R17).  This function is the
 * deterministic part given the DELAYED fast variable xd_j = x_j(t - tau) of every element (xd = x
 * itself when tau = 0); the noise term is added by the integrator (ora_fhn2_rk4).
 * p = {eps, a, sigma, I_app}. */
static void rhs_fhn2(const ora_net* net, const double* y, const double* xd, double* f) {
    const int64_t n = net->n;
    const double eps = net->p[0], a = net->p[1], sigma = net->p[2], Iapp = net->p[3];
    const double* x = y;
    const double* v = y + n;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double Cx = 0.0;
        int64_t links_amount = 0;
        for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e, ++links_amount)
            Cx += xd[net->col_idx[e]] - x[i];
        double s = links_amount > 0 ? sigma / (double)links_amount : 0.0;
        f[i] = (x[i] - x[i] * x[i] * x[i] / 3.0 - v[i] + s * Cx + Iapp) / eps;
        f[n + i] = x[i] + a;
    }
}

/* Hodgkin-Huxley element with the synaptic gating ODE of eq. (1) ("ds_ik/dt =
 * p_ik(U_i, s_ik, n_j)", s_ik "the synaptic conductivity from the k-th to the i-th neuron").
 * Reading R18: p depends on the presynaptic voltage only, so all links leaving element k share
 * one gating variable s_k with first-order kinetics driven by the same sigmoid as rhs_hh:
 *   ds_k/dt = a_s S(V_k) (1 - s_k) - b_s s_k,   S(V) = 1/(1+exp(-(V-theta_syn)/k_syn)),
 *   I_syn,i = (g_syn/Omega_i)(E_syn - V_i) sum_{k in row i} s_k.
 * State SoA [V | m | h | n | s].  p = HH's eleven parameters, then a_s (p[11]), b_s (p[12]). */
static void rhs_hhs(const ora_net* net, const double* y, double* f) {
    const int64_t n = net->n;
    const double gNa = net->p[0], gK = net->p[1], gL = net->p[2];
    const double ENa = net->p[3], EK = net->p[4], EL = net->p[5], C = net->p[6];
    const double gsyn = net->p[7], Esyn = net->p[8], th = net->p[9], ks = net->p[10];
    const double as = net->p[11], bs = net->p[12];
    const double *V = y, *m = y + n, *h = y + 2 * n, *g = y + 3 * n, *sg = y + 4 * n;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double ssum = 0.0;
        int64_t links_amount = 0;
        for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e, ++links_amount)
            ssum += sg[net->col_idx[e]];
        double Isyn = links_amount > 0 ? (gsyn / (double)links_amount) * (Esyn - V[i]) * ssum : 0.0;
        double am, bm, ah, bh, an, bn;
        hh_rates(V[i], &am, &bm, &ah, &bh, &an, &bn);
        double INa = gNa * m[i] * m[i] * m[i] * h[i] * (V[i] - ENa);
        double IK = gK * g[i] * g[i] * g[i] * g[i] * (V[i] - EK);
        double IL = gL * (V[i] - EL);
        f[i] = (net->elem_param[i] - INa - IK - IL + Isyn) / C;
        f[n + i] = am * (1.0 - m[i]) - bm * m[i];
        f[2 * n + i] = ah * (1.0 - h[i]) - bh * h[i];
        f[3 * n + i] = an * (1.0 - g[i]) - bn * g[i];
        f[4 * n + i] = as * (1.0 / (1.0 + exp(-(V[i] - th) / ks))) * (1.0 - sg[i]) - bs * sg[i];
    }
}

/* One full right-hand-side evaluation f(y); y and f are nvar*n SoA.  (FHN2: without delay.) */
int ora_rhs(const ora_net* net, const double* y, double* f) {
    switch (net->model) {
        case ORA_MODEL_FHN2: rhs_fhn2(net, y, y, f); return 0;
        case ORA_MODEL_HHS: rhs_hhs(net, y, f); return 0;
        case ORA_MODEL_KS: rhs_ks(net, y, f); return 0;
        case ORA_MODEL_FHN: rhs_fhn(net, y, f); return 0;
        case ORA_MODEL_HH: rhs_hh(net, y, f); return 0;
        case ORA_MODEL_KSI: rhs_ksi(net, y, f); return 0;
    }
    return -1;
}

/* Gate steady states x_inf(V) = alpha_x/(alpha_x+beta_x) (used to prepare the
 * north-star HH initial condition "gates at steady state"). */
void ora_hh_steady_gates(int64_t n, const double* V, double* m, double* h, double* g) {
    for (int64_t i = 0; i < n; ++i) {
        double am, bm, ah, bh, an, bn;
        hh_rates(V[i], &am, &bm, &ah, &bh, &an, &bn);
        m[i] = am / (am + bm);
        h[i] = ah / (ah + bh);
        g[i] = an / (an + bn);
    }
}

/* Classical 4-stage Runge-Kutta, fixed step (reading R1; the north star
 * prescribes it, the paper's own solvers are adaptive):
 *   k1=f(y); k2=f(y+dt/2 k1); k3=f(y+dt/2 k2); k4=f(y+dt k3);
 *   y <- y + dt/6 (k1 + 2 k2 + 2 k3 + k4).
 * The systems are autonomous, so t is not passed to f. */
int ora_rk4(const ora_net* net, double* y, int64_t n_steps, double dt) {
    int32_t nv = ora_nvar(net->model);
    if (nv < 0) return -1;
    int64_t len = (int64_t)nv * net->n;
    double* buf = (double*)malloc(sizeof(double) * (size_t)len * 5);
    if (!buf) return -2;
    double *k1 = buf, *k2 = buf + len, *k3 = buf + 2 * len, *k4 = buf + 3 * len,
           *tmp = buf + 4 * len;
    for (int64_t s = 0; s < n_steps; ++s) {
        ora_rhs(net, y, k1);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + 0.5 * dt * k1[q];
        ora_rhs(net, tmp, k2);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + 0.5 * dt * k2[q];
        ora_rhs(net, tmp, k3);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + dt * k3[q];
        ora_rhs(net, tmp, k4);
        for (int64_t q = 0; q < len; ++q)
            y[q] = y[q] + (dt / 6.0) * (k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
    }
    free(buf);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Observables (reading R9; the paper names them - "synchronization    */
/* analysis at each output" PAPER.md:416, average frequencies :301,    */
/* coherent/incoherent regions :325 - but gives no formulas).          */
/* ------------------------------------------------------------------ */

/* Phase map theta_i.  KS: phi.  FHN: atan2(v,u).  HH: atan2(n - n_c,
 * (V - V_c)/V_s); pm = {V_c, n_c, V_s}. */
void ora_phase(int32_t model, int64_t n, const double* y, const double* pm, double* theta) {
    for (int64_t i = 0; i < n; ++i) {
        if (model == ORA_MODEL_KS || model == ORA_MODEL_KSI)
            theta[i] = y[i];
        else if (model == ORA_MODEL_FHN || model == ORA_MODEL_FHN2)
            theta[i] = atan2(y[n + i], y[i]);
        else
            theta[i] = atan2(y[3 * n + i] - pm[1], (y[i] - pm[0]) / pm[2]);
    }
}

/* Global Kuramoto order parameter  R e^{i Psi} = (1/N) sum_j e^{i theta_j}. */
void ora_global_order(int64_t n, const double* theta, double* R, double* Psi) {
    double c = 0.0, s = 0.0;
    for (int64_t j = 0; j < n; ++j) {
        c += cos(theta[j]);
        s += sin(theta[j]);
    }
    c /= (double)n;
    s /= (double)n;
    *R = sqrt(c * c + s * s);
    *Psi = atan2(s, c);
}

/* Local order parameter over the coupling neighbourhood plus the element:
 *   R_i = | ( sum_{j in row i} e^{i theta_j} + e^{i theta_i} ) / (Omega_i + 1) |
 * (if the row already holds i, it is not added a second time). */
void ora_local_order(int64_t n, const int64_t* row_ptr, const int32_t* col_idx,
                     const double* theta, double* Rloc) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double c = 0.0, s = 0.0;
        int64_t cnt = 0;
        int has_self = 0;
        for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e, ++cnt) {
            int32_t j = col_idx[e];
            if (j == i) has_self = 1;
            c += cos(theta[j]);
            s += sin(theta[j]);
        }
        if (!has_self) {
            c += cos(theta[i]);
            s += sin(theta[i]);
            ++cnt;
        }
        Rloc[i] = sqrt(c * c + s * s) / (double)cnt;
    }
}

/* ------------------------------------------------------------------ */
/* Accelerated restatement for the LONG statistics runs ONLY           */
/* (last paragraph: "if the box has too few cores, the  */
/* long-run oracle may switch to its own independently written          */
/* factorised/prefix neighbour sum after that variant has been shown    */
/* equal to the direct sum to 1e-13 (A11 norm) on a full-size single    */
/* RHS").  Nothing else uses it: every RHS / trajectory parity test     */
/* compares against ora_rhs / ora_rk4 above.  Written for this file     */
/* alone; it shares nothing with the CUDA library.                      */
/*   KS, KSI: sin(phi_j - phi_i - alpha) = sin phi_j cos(phi_i + alpha) */
/*            - cos phi_j sin(phi_i + alpha): cos/sin once per element, */
/*            then the SAME neighbour loop over row i adds them.        */
/*   HH     : S(V_j) once per element, then the same neighbour loop.    */
/*   FHN    : sum_j (u_j - u_i) = (sum_j u_j) - Omega_i u_i; on a ring   */
/*            (ring_P > 0) the window sum is a difference of prefix     */
/*            sums held in long double.                                 */
/* Pins: tests/test_oracle_dynamics.py::test_fast_variant_* (equal to   */
/* the direct form to 1e-13 on every model/topology); the script        */
/* tests/golden/make_stats_cache.py repeats that check at full size     */
/* before it trusts the variant and stores the discrepancy it saw.      */
/* ------------------------------------------------------------------ */
int ora_rhs_fast(const ora_net* net, const double* y, double* f, int64_t ring_P) {
    const int64_t n = net->n;
    if (net->model == ORA_MODEL_KS || net->model == ORA_MODEL_KSI) {
        const int inertia = net->model == ORA_MODEL_KSI;
        const double K = net->p[0], alpha = net->p[1];
        const double m = inertia ? net->p[2] : 1.0, eps = inertia ? net->p[3] : 0.0;
        double* cs = (double*)malloc(sizeof(double) * 2 * (size_t)n);
        if (!cs) return -2;
        double *c = cs, *s = cs + n;
#pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < n; ++j) { c[j] = cos(y[j]); s[j] = sin(y[j]); }
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double C = 0.0, S = 0.0;
            int64_t links_amount = net->row_ptr[i + 1] - net->row_ptr[i];
            for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e) {
                int32_t j = net->col_idx[e];
                C += c[j];
                S += s[j];
            }
            double der = S * cos(y[i] + alpha) - C * sin(y[i] + alpha);
            if (links_amount > 0) der /= (double)links_amount;
            if (!inertia) f[i] = net->elem_param[i] + K * der;
            else {
                f[i] = y[n + i];
                f[n + i] = (-eps * y[n + i] + net->elem_param[i] + K * der) / m;
            }
        }
        free(cs);
        return 0;
    }
    if (net->model == ORA_MODEL_HH) {
        const double th = net->p[9], ks = net->p[10];
        double* sv = (double*)malloc(sizeof(double) * (size_t)n);
        if (!sv) return -2;
#pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < n; ++j) sv[j] = 1.0 / (1.0 + exp(-(y[j] - th) / ks));
        const double gNa = net->p[0], gK = net->p[1], gL = net->p[2];
        const double ENa = net->p[3], EK = net->p[4], EL = net->p[5], C = net->p[6];
        const double gsyn = net->p[7], Esyn = net->p[8];
        const double *V = y, *mm = y + n, *h = y + 2 * n, *g = y + 3 * n;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double ssum = 0.0;
            int64_t links_amount = net->row_ptr[i + 1] - net->row_ptr[i];
            for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e) ssum += sv[net->col_idx[e]];
            double Isyn = links_amount > 0 ? (gsyn / (double)links_amount) * (Esyn - V[i]) * ssum : 0.0;
            double am, bm, ah, bh, an, bn;
            hh_rates(V[i], &am, &bm, &ah, &bh, &an, &bn);
            double INa = gNa * mm[i] * mm[i] * mm[i] * h[i] * (V[i] - ENa);
            double IK = gK * g[i] * g[i] * g[i] * g[i] * (V[i] - EK);
            double IL = gL * (V[i] - EL);
            f[i] = (net->elem_param[i] - INa - IK - IL + Isyn) / C;
            f[n + i] = am * (1.0 - mm[i]) - bm * mm[i];
            f[2 * n + i] = ah * (1.0 - h[i]) - bh * h[i];
            f[3 * n + i] = an * (1.0 - g[i]) - bn * g[i];
        }
        free(sv);
        return 0;
    }
    if (net->model == ORA_MODEL_FHN) {
        const double eps = net->p[0], a = net->p[1], sigma = net->p[2];
        const double buu = net->p[3], buv = net->p[4], bvu = net->p[5], bvv = net->p[6];
        const double *u = y, *v = y + n;
        long double* pre = NULL;
        if (ring_P > 0) {
            /* pre_u[k] = u_0 + ... + u_{k-1}; the window i-P..i+P (self included, its term is 0)
             * is a difference of two prefix values plus the full-ring total where it wraps */
            pre = (long double*)malloc(sizeof(long double) * 2 * (size_t)(n + 1));
            if (!pre) return -2;
            long double *pu = pre, *pv = pre + n + 1;
            pu[0] = pv[0] = 0.0L;
            for (int64_t k = 0; k < n; ++k) { pu[k + 1] = pu[k] + u[k]; pv[k + 1] = pv[k] + v[k]; }
        }
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double Su, Sv;
            int64_t links_amount = net->row_ptr[i + 1] - net->row_ptr[i];
            if (ring_P > 0) {
                const long double *pu = pre, *pv = pre + n + 1;
                int64_t lo = i - ring_P, hi = i + ring_P + 1;          /* window [lo, hi) */
                long double wu = 0.0L, wv = 0.0L;
                if (lo < 0) { wu += pu[n] - pu[lo + n]; wv += pv[n] - pv[lo + n]; lo = 0; }
                if (hi > n) { wu += pu[hi - n]; wv += pv[hi - n]; hi = n; }
                wu += pu[hi] - pu[lo];
                wv += pv[hi] - pv[lo];
                /* the window holds i itself: sum_{j != i} (u_j - u_i) = W - (2P+1) u_i */
                Su = (double)(wu - (long double)(2 * ring_P + 1) * u[i]);
                Sv = (double)(wv - (long double)(2 * ring_P + 1) * v[i]);
            } else {
                double tu = 0.0, tv = 0.0;
                for (int64_t e = net->row_ptr[i]; e < net->row_ptr[i + 1]; ++e) {
                    int32_t j = net->col_idx[e];
                    tu += u[j];
                    tv += v[j];
                }
                Su = tu - (double)links_amount * u[i];
                Sv = tv - (double)links_amount * v[i];
            }
            double sc = links_amount > 0 ? sigma / (double)links_amount : 0.0;
            f[i] = (u[i] - u[i] * u[i] * u[i] / 3.0 - v[i] + sc * (buu * Su + buv * Sv)) / eps;
            f[n + i] = u[i] + a + sc * (bvu * Su + bvv * Sv);
        }
        free(pre);
        return 0;
    }
    return -1;
}

/* ora_rk4 with ora_rhs_fast in place of ora_rhs (same textbook RK4, same order of operations). */
int ora_rk4_fast(const ora_net* net, double* y, int64_t n_steps, double dt, int64_t ring_P) {
    int32_t nv = ora_nvar(net->model);
    if (nv < 0) return -1;
    int64_t len = (int64_t)nv * net->n;
    double* buf = (double*)malloc(sizeof(double) * (size_t)len * 5);
    if (!buf) return -2;
    double *k1 = buf, *k2 = buf + len, *k3 = buf + 2 * len, *k4 = buf + 3 * len, *tmp = buf + 4 * len;
    for (int64_t s = 0; s < n_steps; ++s) {
        ora_rhs_fast(net, y, k1, ring_P);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + 0.5 * dt * k1[q];
        ora_rhs_fast(net, tmp, k2, ring_P);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + 0.5 * dt * k2[q];
        ora_rhs_fast(net, tmp, k3, ring_P);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + dt * k3[q];
        ora_rhs_fast(net, tmp, k4, ring_P);
        for (int64_t q = 0; q < len; ++q)
            y[q] = y[q] + (dt / 6.0) * (k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
    }
    free(buf);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Dormand-Prince 5(4) with step-size control (the    */
/* solver the paper names first: "a Dormand-Prince solver  */
/* of 3, 5, or 8 order [22] for non-stiff problems").  The paper prints */
/* neither the tableau nor the controller; both are the textbook ones   */
/* of its reference [22] (Hairer, Norsett, Wanner, "Solving Ordinary    */
/* Differential Equations I", the code DOPRI5), reading R15:  */
/*   stages  k1 = f(y)  (first-same-as-last: k1 of a step after an       */
/*           accepted one is k7 of that step),                           */
/*           k_s = f(y + h sum_{j<s} a_sj k_j),  s = 2..7,               */
/*   y5   = y + h sum_j b_j k_j   (b = a_7., the 5th-order solution),    */
/*   e    = h sum_j (b_j - bhat_j) k_j        (bhat: embedded 4th order) */
/*   err  = sqrt( (1/n) sum_i (e_i / (atol + rtol max(|y_i|, |y5_i|)))^2 ) */
/*   accept iff err <= 1;                                                */
/*   h_new = h * min(facmax, max(0.2, 0.9 err^(-1/5))), facmax = 10, and */
/*           1 for the step right after a rejection; err = 0 -> facmax.  */
/*   the last step is shortened to land on t_end exactly                 */
/*           (if t + 1.01 h >= t_end then h = t_end - t).                */
/* The systems are autonomous, so the nodes c_s are not needed.          */
/* Pins (tests/test_oracle_dp5.py): stability polynomial of one step on  */
/* a linear problem (1 + z + ... + z^5/120 + z^6/600, textbook), the     */
/* embedded error of that step, order 5 against a 16x finer run, exact   */
/* for constant RHS, accepted/rejected sequence equal to a scalar DOPRI5 */
/* written out by hand on one FHN element.                               */
/* ------------------------------------------------------------------ */
static const double DP_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5.0, 0, 0, 0, 0, 0},
    {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
static const double DP_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0,
                               -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0};

/* One step of size h from y with k1 given.  Writes y5 (the 5th-order solution), k7 = f(y5) into
 * k[6], and the error vector e.  k = 7 arrays of nvar*n. */
static void dp5_stages(const ora_net* net, const double* y, double h, double** k, double* y5,
                       double* e, double* tmp) {
    const int64_t len = (int64_t)ora_nvar(net->model) * net->n;
    for (int s = 1; s < 7; ++s) {
        double* dst = s == 6 ? y5 : tmp;
        for (int64_t q = 0; q < len; ++q) {
            double acc = 0.0;
            for (int j = 0; j < s; ++j) acc += DP_A[s][j] * k[j][q];
            dst[q] = y[q] + h * acc;
        }
        ora_rhs(net, dst, k[s]);
    }
    for (int64_t q = 0; q < len; ++q) {
        double acc = 0.0;
        for (int j = 0; j < 7; ++j) acc += DP_E[j] * k[j][q];
        e[q] = h * acc;
    }
}

/* A single step of fixed size (no control): y5 and the embedded error vector e (pin hook). */
int ora_dp5_step(const ora_net* net, const double* y, double h, double* y5, double* e) {
    int32_t nv = ora_nvar(net->model);
    if (nv < 0) return -1;
    const int64_t len = (int64_t)nv * net->n;
    double* buf = (double*)malloc(sizeof(double) * (size_t)len * 8);
    if (!buf) return -2;
    double* k[7];
    for (int j = 0; j < 7; ++j) k[j] = buf + j * len;
    ora_rhs(net, y, k[0]);
    dp5_stages(net, y, h, k, y5, e, buf + 7 * len);
    free(buf);
    return 0;
}

/* Integrates from t0 to t_end.  y is advanced in place.  out[0..4] = {accepted steps, rejected
 * steps, last step size used, suggested next step size, t reached}.  h_log (may be NULL) receives
 * the size of every ATTEMPTED step, negative when it was rejected, up to h_log_cap entries.
 * Returns 0, or 1 if max_attempts was exhausted before t_end. */
int ora_dp5(const ora_net* net, double* y, double t0, double t_end, double rtol, double atol,
            double h0, int64_t max_attempts, double* out, double* h_log, int64_t h_log_cap) {
    int32_t nv = ora_nvar(net->model);
    if (nv < 0 || !(h0 > 0.0) || !(t_end >= t0)) return -1;
    const int64_t len = (int64_t)nv * net->n;
    double* buf = (double*)malloc(sizeof(double) * (size_t)len * 10);
    if (!buf) return -2;
    double* k[7];
    for (int j = 0; j < 7; ++j) k[j] = buf + j * len;
    double *y5 = buf + 7 * len, *e = buf + 8 * len, *tmp = buf + 9 * len;
    double t = t0, h = h0, h_used = 0.0;
    int64_t acc_n = 0, rej_n = 0, att = 0;
    int after_reject = 0, rc = 0;
    ora_rhs(net, y, k[0]);
    while (t < t_end) {
        if (att >= max_attempts) { rc = 1; break; }
        int last = 0;
        if (t + 1.01 * h >= t_end) { h = t_end - t; last = 1; }
        dp5_stages(net, y, h, k, y5, e, tmp);
        double s2 = 0.0;
        for (int64_t q = 0; q < len; ++q) {
            double sc = atol + rtol * fmax(fabs(y[q]), fabs(y5[q]));
            double r = e[q] / sc;
            s2 += r * r;
        }
        const double err = sqrt(s2 / (double)len);
        const double facmax = after_reject ? 1.0 : 10.0;
        double fac = err > 0.0 ? 0.9 * pow(err, -0.2) : facmax;
        fac = fmin(facmax, fmax(0.2, fac));
        if (h_log && att < h_log_cap) h_log[att] = err <= 1.0 ? h : -h;
        ++att;
        if (err <= 1.0) {
            t = last ? t_end : t + h;
            h_used = h;
            memcpy(y, y5, sizeof(double) * (size_t)len);
            double* sw = k[0]; k[0] = k[6]; k[6] = sw;      /* first same as last */
            ++acc_n;
            after_reject = 0;
        } else {
            ++rej_n;
            after_reject = 1;
        }
        h *= fac;
    }
    out[0] = (double)acc_n; out[1] = (double)rej_n; out[2] = h_used; out[3] = h; out[4] = t;
    free(buf);
    return rc;
}


/* Dense output of DOPRI5 ("our approach interpolates the solution for dense output", PAPER.md:416;
 * SURVEY.md 8(f).2 "dense output optional").  The continuous extension of the paper's reference [22]
 * (Hairer, Norsett, Wanner, code DOPRI5, routine CONTD5): after an accepted step from (t, y) to
 * (t + h, y5) with stages k1..k7, for theta = (t_out - t)/h in (0, 1]:
 *   r1 = y, r2 = y5 - y, r3 = h k1 - r2, r4 = r2 - h k7 - r3,
 *   r5 = h (d1 k1 + d3 k3 + d4 k4 + d5 k5 + d6 k6 + d7 k7),
 *   y(t + theta h) = r1 + theta (r2 + (1 - theta)(r3 + theta (r4 + (1 - theta) r5)))
 * (fourth-order accurate; equals y at theta = 0 and y5 at theta = 1).  The step control is that of
 * ora_dp5, the steps are NOT shortened to hit the output times (only t_out[n_out-1] = t_end is hit).
 * t_out ascending, t0 < t_out[0]; out = n_out states of nvar*n.  stats as ora_dp5's out. */
static const double DP_D[7] = {-12715105075.0 / 11282082432.0, 0.0, 87487479700.0 / 32700410799.0,
                               -10690763975.0 / 1880347072.0, 701980252875.0 / 199316789632.0,
                               -1453857185.0 / 822651844.0, 69997945.0 / 29380423.0};

int ora_dp5_dense(const ora_net* net, double* y, double t0, int64_t n_out, const double* t_out, double* out,
                  double rtol, double atol, double h0, int64_t max_attempts, double* stats) {
    int32_t nv = ora_nvar(net->model);
    if (nv < 0 || !(h0 > 0.0) || n_out < 1 || !(t_out[0] > t0)) return -1;
    for (int64_t q = 1; q < n_out; ++q) if (!(t_out[q] > t_out[q - 1])) return -1;
    const double t_end = t_out[n_out - 1];
    const int64_t len = (int64_t)nv * net->n;
    double* buf = (double*)malloc(sizeof(double) * (size_t)len * 10);
    if (!buf) return -2;
    double* k[7];
    for (int j = 0; j < 7; ++j) k[j] = buf + j * len;
    double *y5 = buf + 7 * len, *e = buf + 8 * len, *tmp = buf + 9 * len;
    double t = t0, h = h0, h_used = 0.0;
    int64_t acc_n = 0, rej_n = 0, att = 0, next = 0;
    int after_reject = 0, rc = 0;
    ora_rhs(net, y, k[0]);
    while (t < t_end) {
        if (att >= max_attempts) { rc = 1; break; }
        int last = 0;
        if (t + 1.01 * h >= t_end) { h = t_end - t; last = 1; }
        dp5_stages(net, y, h, k, y5, e, tmp);
        double s2 = 0.0;
        for (int64_t q = 0; q < len; ++q) {
            double sc = atol + rtol * fmax(fabs(y[q]), fabs(y5[q]));
            double r = e[q] / sc;
            s2 += r * r;
        }
        const double err = sqrt(s2 / (double)len);
        const double facmax = after_reject ? 1.0 : 10.0;
        double fac = err > 0.0 ? 0.9 * pow(err, -0.2) : facmax;
        fac = fmin(facmax, fmax(0.2, fac));
        ++att;
        if (err <= 1.0) {
            const double t_new = last ? t_end : t + h;
            while (next < n_out && t_out[next] <= t_new) {       /* output times inside this step */
                const double th = last && next == n_out - 1 ? 1.0 : (t_out[next] - t) / h, th1 = 1.0 - th;
                double* o = out + next * len;
                for (int64_t q = 0; q < len; ++q) {
                    const double r2 = y5[q] - y[q], r3 = h * k[0][q] - r2, r4 = r2 - h * k[6][q] - r3;
                    double r5 = 0.0;
                    for (int j = 0; j < 7; ++j) r5 += DP_D[j] * k[j][q];
                    r5 *= h;
                    o[q] = y[q] + th * (r2 + th1 * (r3 + th * (r4 + th1 * r5)));
                }
                ++next;
            }
            t = t_new;
            h_used = h;
            memcpy(y, y5, sizeof(double) * (size_t)len);
            double* sw = k[0]; k[0] = k[6]; k[6] = sw;
            ++acc_n;
            after_reject = 0;
        } else {
            ++rej_n;
            after_reject = 1;
        }
        h *= fac;
    }
    stats[0] = (double)acc_n; stats[1] = (double)rej_n; stats[2] = h_used; stats[3] = h; stats[4] = t;
    free(buf);
    return rc;
}


/* ------------------------------------------------------------------ */
/* Eq. (2) with delay tau and noise D n(t) under fixed-step RK4        */
/* (reading R17).  The paper's own solvers keep       */
/* "data from previous time steps and perform interpolation"           */
/* (PAPER.md:101); with a fixed step that becomes:                     */
/*   tau = m dt, m >= 0 an integer;                                     */
/*   history: x_j and dx_j/dt at the step times t_n (dx/dt = the k1 of  */
/*     that step), m + 2 slots, slot of step q = q mod (m + 2); before  */
/*     the first step every slot holds the initial x with derivative 0  */
/*     (constant initial function);                                     */
/*   the RK4 stages at t_n, t_n + dt/2, t_n + dt/2, t_n + dt see        */
/*     x_j(t_n - tau) = H[n-m],                                          */
/*     x_j(t_n + dt/2 - tau) = cubic Hermite midpoint of H[n-m], H[n-m+1] */
/*        = (xa + xb)/2 + dt/8 (da - db),                               */
/*     x_j(t_n + dt - tau) = H[n-m+1]                                    */
/*     (while n < m the interval [t_n - tau, t_n + dt - tau] lies in     */
/*     t <= 0 and the midpoint is the constant initial value: dx/dt has  */
/*     a jump at t = 0, the stored derivative there is the right one)    */
/*     (m = 0: the stage values themselves, an ordinary coupling);      */
/*   noise: additive Gaussian white noise on y by Euler-Maruyama after  */
/*     the deterministic step, y_i += D sqrt(dt) xi(seed, i, n), with   */
/*     xi from a counter-based generator (ora_gauss) so that any other  */
/*     implementation of the same rule draws the same numbers.          */
/* ------------------------------------------------------------------ */

/* Standard normal deviate number (i, n) of stream `seed`: two 53-bit uniforms from the splitmix64
 * finaliser of reading R8, Box-Muller cosine branch.
 *   a = mix(mix(seed + G (i+1)) + G (2n+1)), b = mix(mix(seed + G (i+1)) + G (2n+2)),
 *   u1 = ((a >> 11) + 1) / 2^53 in (0, 1], u2 = (b >> 11) / 2^53 in [0, 1),
 *   xi = sqrt(-2 ln u1) cos(2 pi u2). */
double ora_gauss(uint64_t seed, int64_t i, int64_t n) {
    const uint64_t G = 0x9E3779B97F4A7C15ULL;
    const uint64_t hi = ora_mix64(seed + G * (uint64_t)(i + 1));
    const uint64_t a = ora_mix64(hi + G * (uint64_t)(2 * n + 1));
    const uint64_t b = ora_mix64(hi + G * (uint64_t)(2 * n + 2));
    const double u1 = ((double)(a >> 11) + 1.0) * (1.0 / 9007199254740992.0);
    const double u2 = (double)(b >> 11) * (1.0 / 9007199254740992.0);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

/* n_steps RK4 steps of ORA_MODEL_FHN2 with delay m dt.  hist_x, hist_d: (m + 2) * n doubles each,
 * owned by the caller and carried from call to call; step0 = number of steps taken before this
 * call (0: the history is initialised here).  D = 0: no noise. */
int ora_fhn2_rk4(const ora_net* net, double* y, int64_t n_steps, double dt, int64_t m, double D,
                 uint64_t seed, int64_t step0, double* hist_x, double* hist_d) {
    if (net->model != ORA_MODEL_FHN2 || m < 0) return -1;
    const int64_t n = net->n, len = 2 * n, S = m + 2;
    double* buf = (double*)malloc(sizeof(double) * (size_t)(5 * len + n));
    if (!buf) return -2;
    double *k1 = buf, *k2 = buf + len, *k3 = buf + 2 * len, *k4 = buf + 3 * len, *tmp = buf + 4 * len;
    double* xd = buf + 5 * len;
    if (step0 == 0)
        for (int64_t q = 0; q < S; ++q)
            for (int64_t i = 0; i < n; ++i) { hist_x[q * n + i] = y[i]; hist_d[q * n + i] = 0.0; }
    for (int64_t st = step0; st < step0 + n_steps; ++st) {
        const int64_t qa = ((st - m) % S + S) % S, qb = ((st - m + 1) % S + S) % S, qn = st % S;
        const double *xa = hist_x + qa * n, *da = hist_d + qa * n;
        const double *xb = hist_x + qb * n, *db = hist_d + qb * n;
        /* stage 1 at t_n */
        for (int64_t i = 0; i < n; ++i) hist_x[qn * n + i] = y[i];       /* x at t_n (qa == qn when m = 0) */
        rhs_fhn2(net, y, m > 0 ? xa : y, k1);
        for (int64_t i = 0; i < n; ++i) hist_d[qn * n + i] = k1[i];      /* dx/dt at t_n */
        /* stages 2, 3 at t_n + dt/2 */
        if (m > 0)
            for (int64_t i = 0; i < n; ++i)      /* st < m: the whole interval lies in t <= 0, constant history */
                xd[i] = st < m ? xa[i] : 0.5 * (xa[i] + xb[i]) + 0.125 * dt * (da[i] - db[i]);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + 0.5 * dt * k1[q];
        rhs_fhn2(net, tmp, m > 0 ? xd : tmp, k2);
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + 0.5 * dt * k2[q];
        rhs_fhn2(net, tmp, m > 0 ? xd : tmp, k3);
        /* stage 4 at t_n + dt */
        for (int64_t q = 0; q < len; ++q) tmp[q] = y[q] + dt * k3[q];
        rhs_fhn2(net, tmp, m > 0 ? xb : tmp, k4);
        for (int64_t q = 0; q < len; ++q)
            y[q] = y[q] + (dt / 6.0) * (k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
        if (D != 0.0) {
            const double amp = D * sqrt(dt);
            for (int64_t i = 0; i < n; ++i) y[n + i] += amp * ora_gauss(seed, i, st);
        }
    }
    free(buf);
    return 0;
}
