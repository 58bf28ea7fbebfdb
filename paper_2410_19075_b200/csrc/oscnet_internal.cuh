// Internal declarations shared by the translation units of liboscnet.so.
// Nothing here is part of the C ABI (include/oscnet.h is).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/oscnet.h"

namespace oscnet {

// ---------------------------------------------------------------- parameters
// Model parameters as passed to kernels (always double; kernels convert to T).
struct ModelParams {
    // KS (and KS with inertia: inv_m = 1/m, damp = eps)
    double K, alpha, sin_a, cos_a, inv_m, damp;
    // FHN
    double inv_eps, a, sigma, buu, buv, bvu, bvv;
    // HH
    double gNa, gK, gL, ENa, EK, EL, inv_C, g_syn, E_syn, theta_syn, inv_k_syn;
    double V_c, n_c, inv_V_s;
    // HHS (gating ODE) and FHN2 (eq. (2): applied current, noise amplitude)
    double a_s, b_s, I_app, noise_D;
    unsigned long long noise_seed;
};

// Topology as seen by kernels.
struct TopoView {
    int32_t kind;          // NET_TOPO_*
    int32_t ndim;
    int32_t nx, ny, nz;    // lattice extents (1 for unused dims)
    int32_t P;             // ring: neighbours per side; lattice: Euclidean radius
    int32_t include_self;
    int32_t noff;          // lattice: number of offsets (= Omega)
    int32_t k_uniform;     // RANDOM_INDEGREE: in-degree; else 0
    int64_t ring_n;        // ring: period (elements per ring; n / batch)
    const int32_t* off;    // lattice: noff x (dx,dy,dz), sorted by (dz,dy,dx)
    const int64_t* row_ptr;
    const int32_t* col_idx;
    // NET_TOPO_COMPRESSED (Alg. 2): common vector, difference table, row references, degree per entry
    const int32_t* cmp_v;
    const int64_t* cmp_dptr;
    const int32_t* cmp_dpos;
    const int32_t* cmp_c;
    const int32_t* cmp_deg;
    int32_t cmp_vlen, cmp_k, cmp_maxdeg;
};

// RK4 in the low-traffic form: four state-sized arrays
// y, Y2, Y3, Y4; no separate accumulator.
//   stage 0: Y2 = y + dt/2 f(y)      stage 1: Y3 = y + dt/2 f(Y2)
//   stage 2: Y4 = y + dt   f(Y3)     stage 3: y  = (Y2 + 2 Y3 + Y4 - y)/3 + dt/6 f(Y4)
//   stage 4 (RHS only): out = f(in)
enum { STAGE_RHS_ONLY = 4 };

struct StageArgs {
    const void* in;   // array the RHS is evaluated on (stencil source)
    const void* y;    // base state
    const void* Y2;
    const void* Y3;
    void* out;
    const void* elem_param;  // omega / I_ext, may be null
    const void* s_in;        // HH fast path: S(V) of `in`
    void* s_out;             // HH fast path: S(V) of `out`
    int64_t n, ld;
    double dt;
    int32_t stage;
};

template <class T>
__device__ __forceinline__ T stage_combine(int stage, T dt, T k, T y, T Y2, T Y3, T Y4in) {
    // Y4in is the value of the stage input at this element (only used in stage 3).
    switch (stage) {
        case 0:
        case 1: return y + (T(0.5) * dt) * k;
        case 2: return y + dt * k;
        case 3: return (Y2 + T(2) * Y3 + Y4in - y) * T(1.0 / 3.0) + (dt * T(1.0 / 6.0)) * k;
        default: return k;
    }
}

// ------------------------------------------------------------------- handle
struct Buffers {
    void *y, *Y2, *Y3, *Y4;       // nvar*ld elements each
    void* elem_param;             // ld elements
    void *s_y, *s_Y2, *s_Y3, *s_Y4;  // HH fast path, ld elements each (else null)
    int32_t* off;                 // lattice offsets
    int64_t* row_ptr;
    int32_t* col_idx;
    int32_t* cmp_v;               // NET_TOPO_COMPRESSED: V, D (ptr, pos), C, degree per table entry
    int64_t* cmp_dptr;
    int32_t* cmp_dpos;
    int32_t* cmp_c;
    int32_t* cmp_deg;
    int32_t* flag;                // device error/validation flag (4 ints)
    // observables
    double* obs_theta_prev;       // n
    double* obs_wind;             // n
    double* obs_ref;              // n (KS: phi at t_a)
    double* obs_vel;              // n
    double* obs_tmp;              // 2n (cos/sin of theta) -- also local-order scratch
    double* obs_loc;              // n
    double* obs_partial;          // reduction partials (4096 doubles)
    double* obs_acc;              // small accumulator block (16 doubles)
    void *hist_x, *hist_d;        // NET_MODEL_FHN2: (delay_steps + 2) slots of ld elements each (x, dx/dt at step times)
    void* scratch;                // method-specific scratch
    size_t scratch_bytes;
};

// launch geometry of the tiled 3D lattice kernels (lattice_fast.cu)
struct Lat3 {
    int32_t nx, ny, nz;
    int32_t TX, S;            // tile: TX columns, S strips of TY rows
    int32_t tiles_x, tiles_y;
    int32_t Lz, nchunks;      // planes per z chunk
    int32_t PW, PH;           // staged plane: (TX+2P) x (S*TY+2P)
    int32_t n_ball;           // lattice points in the ball including the centre
    int32_t include_self;
};

// launch geometry and arguments of the second-generation 3D lattice kernels (lattice_v2.cuh)
constexpr int LAT2_MAXPIECE = 4;

struct Lat2 {
    int32_t nx, ny, nz;
    int32_t QX, SY;            // threads per tile row / strips of TY rows
    int32_t TXt, TYt;          // tile = TXt x TYt outputs
    int32_t tiles_x, tiles_y;
    int32_t Lz, nchunks;
    int32_t PW, PH;            // staged plane: (TXt + 2 HX) x (TYt + 2 P) pairs
    int32_t NS, D;             // ring slots = P + 1 + D, prefetch distance D
    int32_t n_ball, include_self;
};

struct Lat2Args {
    const void* Ein;           // stencil source: pairs [n]
    const void* op0;           // pointwise operands (FHN: pairs; KS: scalars); see kernel
    const void* op1;
    const void* op2;
    const void* omega;         // KS
    void* out;                 // FHN pairs / KS scalar
    void* out2;                // stage 2: Z
    void* Eout;                // KS: pairs of the output state
    double dt;
    int32_t stage;
};

// launch geometry and output pointers of the third-generation 3D lattice kernels (lat3_kernel.cuh)
struct L3Geom {
    int nx, ny, nz;
    int QX, SY;                // consumer threads per tile row / strips of TY rows
    int TXt, TYt;              // tile = TXt x TYt outputs
    int tiles_x, tiles_y, Lz, nchunks;
    int PW, PH;                // staged stencil box: (TXt + 2 HX) x (TYt + 2 P) pairs
    int D;                     // prefetch distance in planes
    int ncw;                   // consumer warps (the producer is warp ncw)
    unsigned st_bytes, st_stride;   // stencil box bytes / ring stride (128-byte multiple)
    unsigned op_bytes, op_stride;   // one operand tile bytes / stride
    long long plane;                // fp64 KS: elements between the cos and the sin plane of E
};

struct L3Ptrs {
    void* out;                 // FHN: padded pairs; KS: plain scalars
    void* out2;                // stage 2: Z
    void* Eout;                // KS: padded (cos, sin) pairs of the output state
};

}  // namespace oscnet

struct net {
    net_desc desc;
    int32_t nvar;
    int32_t esize;
    int64_t n, ld;
    cudaStream_t stream;
    int device;            // ordinal of the device that owns the workspace
    oscnet::ModelParams mp;
    oscnet::TopoView tv;
    oscnet::Buffers b;
    int32_t method;        // NET_METHOD_DIRECT or NET_METHOD_FAST actually in use
    int32_t fast_kind;     // which fast kernel family (internal)
    int64_t nnz;
    int32_t degree_uniform;
    // step driver
    cudaGraphExec_t graph_exec;
    cudaGraph_t graph;
    double graph_dt;
    int32_t graph_steps;
    int64_t graph_kernels;
    int64_t step;
    double t;
    int64_t launches;
    // observed-run results (host copies)
    double stats[8];
    int stats_valid;
    int s_valid;           // HH fast path: s_y consistent with y
    int64_t hist_step;     // NET_MODEL_FHN2: steps taken since the history was reset (net_set_state)
    oscnet::Lat3 lat;      // FAST_LATTICE3D launch geometry
    unsigned lat_grid;
    int lat_threads;
    size_t lat_smem;
    CUtensorMap tmap[4];   // FAST_LATTICE3D_V2: TMA maps of the stencil sources (FHN y,Y2,Y3,Y4; KS E_a,E_b)
    size_t state_bytes;    // bytes of each of y, Y2, Y3, Y4
    oscnet::Lat2 lat2;     // FAST_LATTICE3D_V2 launch geometry
    unsigned lat2_grid;
    int lat2_threads;
    size_t lat2_smem;
    void *E_a, *E_b;       // KS on FAST_LATTICE3D_V2: (cos, sin) pairs of the stage states
    void* ksi_c;           // KSI on FAST_LATTICE3D_V3: coupling term of the stage input (n scalars)
    CUtensorMap tm3_st[4]; // FAST_LATTICE3D_V3: stencil maps (FHN y,Y2,Y3,Y4; KS E_a,E_b)
    CUtensorMap tm3_op[4]; // operand maps (FHN y,Y2 centre boxes; KS y,Y2,Y3,omega scalars)
    oscnet::L3Geom lat3[6]; // per stage (0-3, RHS, local order parameter)
    unsigned lat3_grid[6];
    int lat3_threads[6];
    size_t lat3_smem[6];
    char cb_geom[96];      // FAST_CSR_BLOCKED: CbGeom (csr_blocked.cu)
    unsigned cb_grid;
    int32_t cb_pair;       // 1 = pair form of the blocked CSR kernel (each CTA streams half of the s blocks)
    int32_t cb_es;         // entries staged in shared memory
    size_t cb_smem;
    int32_t l3_force_tx, l3_force_sy, l3_force_ctas;   // FAST_LATTICE3D_V3: tile chosen by the autotuner (0 = by score)
    int32_t l3_force_tail;   // FAST_LATTICE3D_V3: -1 = chunk-aligned grid only, no tail of spans (autotuner)
    int32_t ks_planar;     // 1 = KS exchange fields E_a / E_b are two planes (cos | sin), not pairs (fp64 on FAST_LATTICE3D_V3)
    int32_t pairs;         // 1 = state arrays are ghost-padded interleaved pairs (FHN on FAST_LATTICE3D_V2)
    char err[512];
};

namespace oscnet {

// error helpers -------------------------------------------------------------
int32_t set_err(net* h, int32_t code, const char* fmt, ...);
int32_t cuda_err(net* h, cudaError_t e, const char* what);
#define OSC_CUDA(h, call)                                            \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return oscnet::cuda_err(h, e_, #call); \
    } while (0)

// topology.cu ---------------------------------------------------------------
int32_t topo_lattice_noff(int ndim, int P, int include_self);
int32_t topo_build(net* h);   // fills workspace topology from h->desc
int32_t topo_expand(net* h, int64_t row_begin, int64_t row_count, int64_t* d_row_ptr,
                    int32_t* d_col_idx);  // device destinations

// direct.cu -----------------------------------------------------------------
int32_t direct_stage(net* h, const StageArgs& a);
int32_t hh_compute_s(net* h, const void* V, void* s);     // s = S(V)
int32_t hh_steady_gates(net* h);

// csr_fast.cu / lattice_fast.cu / ring_fast.cu ------------------------------
enum { FAST_NONE = 0, FAST_CSR_WARP = 1, FAST_LATTICE3D = 2, FAST_RING_FHN = 3, FAST_RING_KS = 4,
       FAST_LATTICE3D_V2 = 5, FAST_LATTICE3D_V3 = 6, FAST_CSR_BLOCKED = 7 };
int32_t fast_select(const net_desc* d);                   // FAST_* available for this desc
size_t fast_scratch_bytes(const net_desc* d, int32_t fast_kind);
size_t fast_state_bytes(const net_desc* d, int32_t fast_kind);   // 0 = the default nvar*ld elements
int32_t fast_prepare(net* h);                             // once, at the end of net_create
int32_t fast_stage(net* h, const StageArgs& a);
int32_t fast_integrate(net* h, int64_t n_steps, double dt, bool* handled);  // persistent kernels
int32_t fast_refresh_exchange(net* h, const void* state);   // exchange fields of `state` (nullptr: of y, after set_state)
int32_t pairs_pack(net* h, const void* soa, void* pairs);    // SoA [2][ld] -> padded pairs (+ ghosts)
int32_t pairs_unpack(net* h, const void* pairs, void* soa);

// observables.cu ------------------------------------------------------------
int32_t obs_phase(net* h, const void* state, double* d_theta);
int32_t ring_probe_latency(net* h, double* out4);   // ring_fast.cu
int32_t ring_run_observed(net* h, int64_t n_steps, double dt, int64_t obs_every, int64_t s_a, bool* handled);
int32_t probe_peaks(net* h, double* out8);          // probe.cu
// delay.cu (NET_MODEL_FHN2: eq. (2) with delay and noise)
int32_t delay_stage(net* h, const StageArgs& a);
int32_t delay_reset_history(net* h);
// adaptive.cu (Dormand-Prince 5(4)) and its helpers in api.cu
size_t adaptive_workspace_bytes(const net* h);
int32_t adaptive_integrate(net* h, double t_end, double rtol, double atol, double h0, int64_t max_attempts,
                           void* d_work, size_t work_bytes, double* out5);
int32_t adaptive_integrate_dense(net* h, int64_t n_out, const double* t_out, void* d_out, double rtol, double atol, double h0,
                                 int64_t max_attempts, void* d_work, size_t work_bytes, double* out5);
int32_t state_to_external(net* h, void* d_dst);
int32_t state_from_external(net* h, const void* d_src);
int32_t rhs_at(net* h, const void* d_x, void* d_k);
int32_t obs_global_order(net* h, const double* d_theta, double* d_out2);  // {R, Psi}
int32_t obs_replica_order(net* h, const double* d_theta, double* d_out);  // {R_r, Psi_r} per replica of the batch
int32_t obs_local_order(net* h, const double* d_theta, double* d_out);
bool lattice_v3_has_local_order(const net* h);                 // lattice_v2.cu: ball-sum form of the local order parameter
int32_t lattice_v3_local_order(net* h, double* d_out);
int32_t obs_window_begin(net* h);
int32_t obs_window_sample(net* h, int first);
int32_t obs_window_finish(net* h, double t_a, double t_b, int64_t n_samples);

inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

}  // namespace oscnet
