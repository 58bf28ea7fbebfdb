/*
 * oscnet.h -- C ABI of the B200-native coupled-oscillator RK4 hot path of
 * arXiv:2410.19075 (Sudakov & Maistrenko, "Parallelization of Network Dynamics
 * Computations in Heterogeneous Distributed Environment").
 *
 * The library integrates N coupled oscillators with fixed-step classical RK4.
 * Each right-hand-side evaluation is "local vector field + coupling sum over the
 * in-neighbours the topology allows" (Alg. 1),
 * for the three model classes of Sec. II: Hodgkin-Huxley type (eq. (1),
 * PAPER.md:48-60), FitzHugh-Nagumo (eq. (2)) and
 * Kuramoto-Sakaguchi phase oscillators (eq. (3)), on the coupling
 * topologies of Sec. IV: ring, 2D/3D periodic lattice with
 * Euclidean radius P or an arbitrary runtime graph
 * given as CSR.  "Integration ... requires the runtime
 * specification of initial values for dynamical variables, model parameters,
 * and the coupling topology of the network": these are exactly
 * the arguments of net_create / net_set_state / net_set_param_array.
 *
 * Conventions
 *  - Every function returns an int32_t status: NET_OK or a negative NET_ERR_*.
 *    Nothing throws, aborts or exits.  net_last_error() gives the message of the
 *    last failing call on that handle (or of the last failing net_create /
 *    net_workspace_bytes when called with NULL).
 *  - The library never allocates device memory.  All device storage (state,
 *    RK4 stages, topology, scratch) lives in the caller's workspace, whose size
 *    net_workspace_bytes() reports.  The handle is a small host object.
 *  - The CUDA stream is borrowed.  Every call enqueues its work on that stream.
 *    Calls whose source/destination is a HOST pointer synchronise the stream
 *    before returning; calls with DEVICE pointers are stream-ordered and
 *    asynchronous.  Asynchronous CUDA faults surface at the next synchronising
 *    call as NET_ERR_CUDA.
 *  - State layout: structure of arrays [nvar][n], element type = the dtype of
 *    the net (float or double), contiguous (variable v of element i at
 *    v*n + i).  nvar: KS 1 (phi); FHN 2 (u, v); HH 4 (V, m, h, n); KSI 2 (phi, psi); FHN2 2 (x, y);
 *    HHS 5 (V, m, h, n, s).
 *  - Element numbering of lattices: site (i,j,k) is element k*nx*ny + j*nx + i
 *    (PAPER.md:309 "jN1+i", :311 "kN1^2+jN1+i").
 *  - CSR orientation: row i lists the elements j that influence i
 *    (L_ij = 1 iff the j-th oscillator influences the i-th).
 */
#ifndef OSCNET_H
#define OSCNET_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct net net_t;

enum {
    NET_OK = 0,
    NET_ERR_INVALID = -1,     /* null pointer, bad enum, bad size, 2*radius >= extent, ... */
    NET_ERR_SIZE = -2,        /* workspace too small or misaligned (needs 256-byte alignment) */
    NET_ERR_TOPOLOGY = -3,    /* CSR not monotone / index out of range / self-loop where forbidden */
    NET_ERR_CUDA = -4,        /* a CUDA call failed; message holds cudaGetErrorString */
    NET_ERR_UNSUPPORTED = -5  /* valid request this build does not implement (e.g. NET_METHOD_FAST on a 2D lattice) */
};

enum { NET_MODEL_KS = 0, NET_MODEL_FHN = 1, NET_MODEL_HH = 2,
       NET_MODEL_KSI = 3,  /* KS with inertia, eq. (3) in full */
       NET_MODEL_FHN2 = 4, /* FHN exactly as eq. (2): x-only coupling, delay, noise, I_app (DIRECT kernels) */
       NET_MODEL_HHS = 5   /* HH with the synaptic gating ODE of eq. (1) (DIRECT kernels) */ };
enum { NET_TOPO_RING = 0, NET_TOPO_LATTICE = 1, NET_TOPO_CSR = 2, NET_TOPO_RANDOM_INDEGREE = 3,
       NET_TOPO_COMPRESSED = 4 /* differentially compressed coupling matrix, Alg. 2 */ };
enum { NET_F32 = 0, NET_F64 = 1 };

/* How the coupling sum is evaluated.  DIRECT = one term per neighbour, gathered
 * from global memory (the formulation of Alg. 1).  FAST = the rewrite for that
 * model/topology that is exact in real arithmetic: factorised sine + tiled
 * window sums on lattices, prefix sums on rings, warp-per-row gathers of
 * precomputed synaptic activations on graphs.  AUTO = FAST where one exists. */
enum { NET_METHOD_AUTO = 0, NET_METHOD_DIRECT = 1, NET_METHOD_FAST = 2 };

enum { NET_PARAM_OMEGA = 0, NET_PARAM_IEXT = 1 };

enum {
    NET_OBS_PHASE = 0,               /* theta[n] of the current state, dtype double */
    NET_OBS_GLOBAL_ORDER = 1,        /* double[2] = {R, Psi}: R e^{i Psi} = (1/N) sum_j e^{i theta_j} */
    NET_OBS_LOCAL_ORDER = 2,         /* double[n]: R_i over the coupling neighbourhood plus i */
    NET_OBS_MEAN_PHASE_VELOCITY = 3, /* double[n] over the window of net_integrate_observed */
    NET_OBS_STATS = 4,               /* double[8], see net_integrate_observed */
    NET_OBS_REPLICA_ORDER = 5        /* double[2*batch] = {R_r, Psi_r} of every replica r of a batch (batch = 1:
                                      * the same as NET_OBS_GLOBAL_ORDER) */
};

/* Kuramoto-Sakaguchi, eq. (3) with m=0, eps=1, mu=K/Omega_i:
 *   dphi_i/dt = omega_i + (K/Omega_i) sum_{j in row i} sin(phi_j - phi_i - alpha).
 * omega_i = omega0 for all i until net_set_param_array(NET_PARAM_OMEGA). */
typedef struct {
    double K, alpha, omega0;
} net_ks_params;

/* Kuramoto-Sakaguchi with inertia, eq. (3) in full (the model of the paper's performance
 * tests), as a first-order system in (phi, psi = dphi/dt), nvar = 2:
 *   dphi_i/dt = psi_i
 *   dpsi_i/dt = ( -eps psi_i + omega_i + (K/Omega_i) sum_{j in row i} sin(phi_j - phi_i - alpha) ) / m
 * (K/Omega_i = the paper's mu; omega_i = omega0 until net_set_param_array(NET_PARAM_OMEGA), 0 in the
 * paper).  State [phi | psi].  NET_METHOD_FAST: rings (and batches of rings) run the persistent
 * prefix-sum kernel, 3D balls of radius 2 / 4 / 6 the field-split lattice kernels, graphs the
 * warp-per-row gathers; 1D / 2D lattices are served by NET_METHOD_DIRECT (the per-link form of Alg. 1). */
typedef struct {
    double K, alpha, m, eps, omega0;
} net_ksi_params;

/* FitzHugh-Nagumo, eq. (2) with rotated 2x2 diffusive coupling:
 *   eps du_i/dt = u_i - u_i^3/3 - v_i + (sigma/Omega_i) sum_j [b_uu (u_j-u_i) + b_uv (v_j-v_i)]
 *       dv_i/dt = u_i + a           + (sigma/Omega_i) sum_j [b_vu (u_j-u_i) + b_vv (v_j-v_i)]
 *   (b_uu, b_uv, b_vu, b_vv) = (cos phi, sin phi, -sin phi, cos phi). */
typedef struct {
    double eps, a, sigma, phi;
} net_fhn_params;

/* FitzHugh-Nagumo exactly as the paper prints it, eq. (2), nvar = 2, state [x | y]:
 *   eps dx_i/dt = x_i - x_i^3/3 - y_i + (sigma/Omega_i) sum_{j in row i} (x_j(t - tau) - x_i) + I_app
 *       dy_i/dt = x_i + a + D n_i(t)
 * (uniform coupling strength s_ij = sigma/Omega_i).  Under the fixed-step RK4 of net_integrate
 * (reading R17): tau = net_desc.delay_steps * dt; the library keeps x and dx/dt of the last
 * delay_steps + 2 step times in the workspace ("maintaining data from previous time steps and
 * performing interpolation") and the half-step stages read the cubic Hermite midpoint;
 * before the first step the history is the constant initial x (net_set_state resets it).  The noise
 * is additive Gaussian white noise on y by Euler-Maruyama: after every step
 * y_i += D sqrt(dt) xi(seed, i, step) with xi from the counter-based generator of reading R17
 * (splitmix64 finaliser, Box-Muller), so that runs are reproducible and comparable across
 * implementations.  net_eval_rhs gives the deterministic right-hand side without delay.
 * net_integrate_adaptive is refused while delay_steps > 0 or D != 0. */
typedef struct {
    double eps, a, sigma, I_app, D;
    uint64_t seed;
} net_fhn2_params;

/* Hodgkin-Huxley type element, eq. (1), standard squid-axon
 * channels and an instantaneous sigmoidal synapse (mV, ms, uA/cm^2, mS/cm^2, uF/cm^2):
 *   C dV_i/dt = I_ext,i - gNa m^3 h (V-ENa) - gK n^4 (V-EK) - gL (V-EL)
 *               + (g_syn/Omega_i)(E_syn - V_i) sum_{j in row i} S(V_j),
 *   S(V) = 1/(1+exp(-(V-theta_syn)/k_syn)),  dx/dt = alpha_x(V)(1-x) - beta_x(V) x.
 * I_ext,i = I_ext0 until net_set_param_array(NET_PARAM_IEXT).
 * (V_c, n_c, V_s) define the phase map theta = atan2(n - n_c, (V - V_c)/V_s). */
typedef struct {
    double gNa, gK, gL, ENa, EK, EL, C, g_syn, E_syn, theta_syn, k_syn;
    double I_ext0;
    double V_c, n_c, V_s;
} net_hh_params;

/* Hodgkin-Huxley element with the synaptic gating ODE of eq. (1) ("ds_ik/dt = p_ik(U_i, s_ik, n_j)",
 * PAPER.md:54), nvar = 5, state [V | m | h | n | s].  Reading R18: the kinetics depend on the
 * presynaptic voltage only, so all links leaving element k share one gating variable s_k:
 *   ds_k/dt = a_s S(V_k)(1 - s_k) - b_s s_k,  I_syn,i = (g_syn/Omega_i)(E_syn - V_i) sum_{k in row i} s_k
 * (S the sigmoid of net_hh_params; everything else as NET_MODEL_HH).  net_hh_steady_gates also sets
 * s to its steady state a_s S/(a_s S + b_s). */
typedef struct {
    net_hh_params hh;
    double a_s, b_s;
} net_hhs_params;

/* Coupling topology (static during a run).
 *  RING:    n elements on a circle, each coupled to `radius` neighbours on both sides.
 *  LATTICE: ndim (1..3) periodic lattice extent[0] x extent[1] x extent[2] (x fastest),
 *           coupled to all sites with squared Euclidean distance <= radius^2.
 *           2*radius < every used extent is required (no site may be reached twice).
 *  CSR:     row_ptr[n+1] (int64), col_idx[nnz] (int32); host or device pointers
 *           (ptrs_are_device); copied into the workspace by net_create.
 *  RANDOM_INDEGREE: every row has exactly in_degree distinct sources != i, drawn by the
 *           integer counter-based rule of DESIGN.md reading R8 from `seed`; built on the device.
 *  COMPRESSED: the differentially compressed matrix of Alg. 2 (`compressed`, from net_compress_csr
 *           or built by the caller).  The device keeps V, D and the n row references -- O(max(BK, n))
 *           memory -- and every stage EXTRACTs rows on the fly: rows whose difference
 *           is empty are the common pattern shifted by i (offset loop, no per-row data); the others
 *           merge V with their table entry ("lattice with defects").  Served by the per-link DIRECT
 *           kernels.
 *  include_self (ring/lattice): also count the centre as a link (then Omega = 2P+1 / 33 / 257,
 *           the link counts the paper prints). */
/* Differentially compressed coupling matrix (Alg. 2), on position sets instead
 * of bit vectors: the common vector V = row 0; for every row i the difference
 * d_i = XOR(ROL(L_i, i), V) (ROL moves the bit at position j to (j - i) mod n); the table D of the
 * distinct differences; C_i = the entry of D that equals d_i.  EXTRACT: row i = the positions
 * (p + i) mod n for p in XOR(V, D[C_i]).  "A full mesh topology has a common vector with all bits
 * set and a difference table with a single entry having all bits unset".
 * All arrays are HOST memory; positions are sorted ascending within V and within each entry. */
typedef struct {
    int64_t n;             /* rows (elements) */
    int64_t v_len;         /* set bits of the common vector */
    const int32_t* v_pos;  /* [v_len] */
    int64_t k;             /* entries of the difference table */
    const int64_t* d_ptr;  /* [k + 1] */
    const int32_t* d_pos;  /* [d_ptr[k]] */
    const int32_t* c;      /* [n] row -> entry of the table */
} net_compressed;

/* COMPRESS of Alg. 2 on the host (done once per matrix, as in the paper: "performed only once",
 * PAPER.md:173): rows given as CSR (host pointers; rows need not be sorted).  The result is owned
 * by the library until net_compressed_free; net_create copies what it needs into the workspace.
 * Cost O(nnz) expected (hashed table lookup). */
int32_t net_compress_csr(int64_t n, const int64_t* row_ptr, const int32_t* col_idx, net_compressed** out);
int32_t net_compressed_free(net_compressed* c);

typedef struct {
    int32_t kind;
    int32_t ndim;
    int64_t extent[3];
    int32_t radius;
    int32_t include_self;
    const int64_t* row_ptr;
    const int32_t* col_idx;
    int64_t nnz;
    int32_t ptrs_are_device;
    int32_t in_degree;
    uint64_t seed;
    const net_compressed* compressed;   /* NET_TOPO_COMPRESSED: the matrix (host); else NULL */
} net_topology;

typedef struct {
    int32_t model;  /* NET_MODEL_*  */
    int32_t dtype;  /* NET_F32 | NET_F64: storage and arithmetic type of the state */
    int64_t n;      /* number of elements of ONE net (64-bit) */
    int32_t batch;  /* >= 1: independent replicas of the net integrated together ("a large number of
                     * network instances simultaneously"), each with its own state and
                     * per-element parameters.  Every array that is [..][n] for batch = 1 becomes
                     * [..][batch][n] (replica-major, n contiguous); element ids in net_get_topology
                     * and the observables run over 0 .. batch*n - 1 (the coupling matrix of the batch
                     * is block diagonal; global observables are ensemble values).  The topology
                     * describes ONE replica.  Rings of <= 2048 elements run one CTA of the persistent
                     * kernel per replica (FAST); batches of lattices and graphs run the per-link DIRECT
                     * kernels; NET_TOPO_COMPRESSED is not batched (NET_ERR_UNSUPPORTED).
                     * n * batch <= 2^31 - 1. */
    int32_t method; /* NET_METHOD_* */
    net_topology topo;
    int32_t delay_steps; /* NET_MODEL_FHN2: tau = delay_steps * dt (0 = no delay); else 0 */
    int32_t reserved_;
} net_desc;

/* Bytes of device workspace net_create needs for this description (pure function). */
int32_t net_workspace_bytes(const net_desc* desc, size_t* bytes);

/* Builds the network: validates, lays out the workspace, builds the topology on the device
 * (offset tables / CSR / random graph) and zeroes the state.  `params` points to the
 * net_*_params struct of desc->model (params_bytes = its sizeof).  d_workspace: device memory,
 * 256-byte aligned, >= net_workspace_bytes; owned by the caller and must outlive the handle.
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  On failure *out is NULL.
 * Cost: 3D lattice nets of >= 2^19 elements on the tiled kernels time the ten best-scoring tiles at
 * three pipeline depths on one RK4 step each (about 500 launches on zeroed buffers, 0.1 - 1 s) and keep
 * the fastest; the arithmetic of every output is the same for every tile, so results do not depend on
 * the pick (tests/test_gpu_round2.py::test_lattice_tiles_give_identical_bits).  The pick is reported
 * by net_get_launch_config.  Environment: OSCNET_NO_AUTOTUNE = take the best-scoring tile untimed;
 * OSCNET_LAT3 = "tile_x,strips,planes_per_chunk,depth,ctas" = that geometry. */
int32_t net_create(const net_desc* desc, const void* params, size_t params_bytes,
                   void* d_workspace, size_t workspace_bytes, void* cuda_stream, net_t** out);

/* Frees the host handle (and its CUDA graph); the workspace stays with the caller. */
int32_t net_destroy(net_t* net);

/* Copies a full state [nvar][n] (dtype of the net) into / out of the net ("runtime specification
 * of initial values"; restart from any saved state).  Resets nothing
 * else; the time and step counter are kept (net_set_time changes them). */
int32_t net_set_state(net_t* net, const void* src, int32_t src_is_device);
int32_t net_get_state(net_t* net, void* dst, int32_t dst_is_device);

/* Per-element parameter array [n] in the dtype of the net: NET_PARAM_OMEGA (KS) or
 * NET_PARAM_IEXT (HH) ("model parameters" specified at run time). */
int32_t net_set_param_array(net_t* net, int32_t which, const void* src, int32_t src_is_device);

/* HH only: sets m, h, n of every element to the steady state x_inf(V_i) of its current V
 * (the north-star initial condition "gates at steady state"). */
int32_t net_hh_steady_gates(net_t* net);

/* Advances the state by n_steps classical RK4 steps of size dt (enqueued, asynchronous).  The
 * integrator is BASELINE.json's (reading R1: the paper itself lists only adaptive / stiff solvers,
 * PAPER.md:99; "the integrator outputs ... values of dynamical variables at specified time moments",
 * call it once per output interval):
 *   k1=f(y); k2=f(y+dt/2 k1); k3=f(y+dt/2 k2); k4=f(y+dt k3); y += dt/6 (k1+2k2+2k3+k4).
 * Every stage is one fused kernel (coupled RHS + stage update); steps are replayed from a
 * captured CUDA graph. */
int32_t net_integrate(net_t* net, int64_t n_steps, double dt);

/* net_integrate plus the long-run statistics of DESIGN.md reading R9 ("synchronization analysis at
 * each output"; average frequencies PAPER.md:301; coherent / incoherent regions
 * the paper names the observables and gives no formulas): samples after steps
 * obs_every, 2*obs_every, ..., n_steps (n_steps % obs_every == 0); the window is the samples
 * with step >= n_steps/2.  Afterwards NET_OBS_STATS gives double[8] =
 * {mean R, std R (population), mean_i R_loc,i at the last sample, mean_i and std_i of the mean
 *  phase velocity over the window, number of samples, t_a, t_b} and
 * NET_OBS_MEAN_PHASE_VELOCITY the per-element velocities. */
int32_t net_integrate_observed(net_t* net, int64_t n_steps, double dt, int64_t obs_every);

/* Adaptive integration from the net's current time to t_end with the Dormand-Prince 5(4) pair and
 * step-size control on the device -- the solver the paper recommends first ("a
 * Dormand-Prince solver of 3, 5, or 8 order [22] for non-stiff problems").  The paper prints neither
 * tableau nor controller; both are the textbook DOPRI5 of its reference [22] (reading R15):
 *   err = sqrt(mean_i (e_i / (atol + rtol max(|y_i|, |y5_i|)))^2), accept iff err <= 1,
 *   h <- h min(facmax, max(0.2, 0.9 err^(-1/5))), facmax = 10 (1 right after a rejection),
 *   first-same-as-last, the last step cut to land on t_end exactly.
 * h0 > 0 is the first step tried.  d_work: device memory, 256-byte aligned, at least
 * net_adaptive_workspace_bytes (10 state-sized vectors), owned by the caller, free to reuse
 * afterwards.  out5 (host) = {accepted steps, rejected steps, last step used, next step suggested,
 * time reached}.  The error norm, the decision and the next step are computed on the device; the
 * host reads the control block once per 8 attempts.  Synchronises the stream.  Returns
 * NET_ERR_INVALID (state and time as reached) when max_attempts is exhausted before t_end.
 * Dense output: net_integrate_adaptive_dense below. */
int32_t net_adaptive_workspace_bytes(net_t* net, size_t* bytes);
int32_t net_integrate_adaptive(net_t* net, double t_end, double rtol, double atol, double h0,
                               int64_t max_attempts, void* d_work, size_t work_bytes, double* out5);

/* net_integrate_adaptive with dense output ("the integrator outputs ... values of dynamical variables
 * at specified time moments"; "our approach interpolates the solution for dense output",
 * PAPER.md:416): the states at the strictly ascending HOST times t_out[0 .. n_out), t_out[0] > the
 * net's time, are written to d_out [n_out][nvar][n] (DEVICE, dtype of the net); the run ends at
 * t_out[n_out - 1].  Interpolant: the continuous extension of DOPRI5 (routine CONTD5 of the paper's
 * reference [22]; fourth order, exact at both ends of a step), evaluated on the device right after
 * each accepted step.  The output times never shorten a step: the step sequence is that of
 * net_integrate_adaptive.  d_work: at least net_adaptive_workspace_bytes + 8 n_out rounded up to 256. */
int32_t net_integrate_adaptive_dense(net_t* net, int64_t n_out, const double* t_out, void* d_out,
                                     double rtol, double atol, double h0, int64_t max_attempts,
                                     void* d_work, size_t work_bytes, double* out5);

/* One right-hand-side evaluation f(y) at the current state, [nvar][n] in the dtype of the net:
 * the paper's Calculate(t, y, der) of Alg. 1 for all elements at once
 * (parity hook; the systems are autonomous, so t is not an argument). */
int32_t net_eval_rhs(net_t* net, void* dst, int32_t dst_is_device);

/* Observables of the current state (or of the last net_integrate_observed window), always
 * double; sizes under NET_OBS_*.  Definitions: DESIGN.md reading R9. */
int32_t net_observables(net_t* net, int32_t what, void* dst, int32_t dst_is_device);

/* Expands rows [row_begin, row_begin+row_count) of the topology to canonical CSR (row i = the
 * elements that influence i; lattice rule PAPER.md:309-313): each row
 * sorted ascending, row_ptr[row_count+1] relative to the range (parity hook; bit-exact
 * against the oracle). */
int32_t net_get_topology(net_t* net, int64_t row_begin, int64_t row_count, int64_t* row_ptr,
                         int32_t* col_idx, int32_t dst_is_device);

/* nnz of the whole topology and the in-degree if every row has the same one (else -1). */
int32_t net_get_degree(net_t* net, int64_t* nnz, int32_t* uniform_degree);

int32_t net_get_time(net_t* net, double* t, int64_t* step);
int32_t net_set_time(net_t* net, double t, int64_t step);

/* Number of kernels this handle has launched (graph replays count their kernel nodes) and
 * the method actually in use (NET_METHOD_DIRECT or NET_METHOD_FAST). */
int32_t net_get_counters(net_t* net, int64_t* kernel_launches, int32_t* method_in_use);

/* Which kernel family serves the fused RHS + RK4 stages of this net (diagnostic; DESIGN.md
 * section 5): NET_FAMILY_DIRECT 0 (Alg. 1 form), CSR_WARP 1, LATTICE3D 2,
 * RING (persistent, FHN 3 / KS 4), LATTICE3D_V2 5, LATTICE3D_V3 6, CSR_BLOCKED 7. */
int32_t net_get_kernel_family(net_t* net, int32_t* family);

/* Launch geometry of the stage kernel in use (diagnostic; the lattice tile is picked by a timing
 * pass inside net_create for nets of >= 2^19 elements, so a bench line should print it).  out8 =
 * {kernel family, tile x, tile y, z planes per chunk, prefetch depth, grid, threads, dynamic shared
 * memory in bytes} of RK4 stage 1; entries a family does not have are 0. */
int32_t net_get_launch_config(net_t* net, int32_t* out8);

/* Blocks until the stream is idle; returns NET_ERR_CUDA if anything failed asynchronously. */
int32_t net_synchronize(net_t* net);

/* Message of the last error on this handle (NULL: of the last failed handle-less call).
 * The string is owned by the library and valid until the next call on the same handle. */
const char* net_last_error(const net_t* net);

/* Diagnostic: latencies of the primitives one stage of a latency-bound (ring) net chains, measured on
 * the net's stream with the net's scratch memory ("fraction of a measured latency
 * model").  out4 (host, microseconds each) = {grid barrier over the CTAs this net's persistent kernel
 * uses (0 for single-CTA nets), one dependent load served by L2, one 256-thread block scan of two
 * doubles, one dependent fp64 sincos}.  Synchronises the stream; the state is not touched. */
int32_t net_probe_latency(net_t* net, double* out4);

/* Diagnostic: peak microbenchmarks on the net's device and stream (the
 * denominators of the ALU- and gather-bound rooflines of SURVEY.md 8(d)).  out8 (host) =
 *   [0] FFMA, [1] add.f32x2, [2] DFMA, [3] MUFU.EX2 thread-instructions per second / 1e9
 *       (8 independent chains per thread, 8 CTAs of 256 threads per SM),
 *   [4] shared-memory read bandwidth in GB/s (conflict-free LDS.128),
 *   [5] independent random 8-byte loads per second / 1e9 from an L2-resident array of out8[6] bytes
 *       (what the gathers of a CSR stage do; the array is min(8 MB, one state array)),
 *   [7] SM clock in MHz as seen by clock64() during the probes.
 * Uses the stage array Y4 (rewritten by every step before it is read) and synchronises the stream;
 * y, the time and the topology are not touched. */
int32_t net_probe_peaks(net_t* net, double* out8);

/* The global order parameter without a handle, a workspace or any allocation: for callers that may
 * not call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 *   R e^{i Psi} = (1/N) sum_j e^{i theta_j}   (reading R9), as NET_OBS_GLOBAL_ORDER.
 * d_theta (DEVICE, caller-owned): n phases of `dtype` (NET_F32 / NET_F64); the sum is in double.
 * d_out2 (DEVICE, caller-owned): double[2] = {R, Psi}, written when the work on `stream` (a cudaStream_t
 * of the CURRENT device, NULL = default stream) completes; the call does not synchronise.
 * The block partials live in one static device array of 262400 bytes that every GPU loading the
 * library holds until exit: n <= NET_NOALLOC_MAX_N, larger n returns NET_ERR_SIZE and launches nothing
 * (message: net_last_error(NULL)).  Every call on a device shares that array, so calls that overlap on
 * the GPU (different streams, graphs replayed concurrently) race: serialise them.  The call enqueues one
 * 256-byte cudaMemsetAsync (the completion ticket must start at zero) and one kernel; it calls no
 * cudaMalloc, cudaFree or allocating library routine.  The first call on each device also resolves the
 * array's device address (cudaGetSymbolAddress): make that one outside stream capture.
 * Errors: NET_ERR_INVALID (NULL pointer, n < 1, bad dtype), NET_ERR_SIZE, NET_ERR_CUDA. */
#define NET_NOALLOC_MAX_N 134217728LL /* 2^27 */
int32_t net_order_parameter_noalloc(const void* d_theta, int64_t n, int32_t dtype, double* d_out2, void* stream);

/* "oscnet <major>.<minor> sm_100a" */
const char* net_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OSCNET_H */
