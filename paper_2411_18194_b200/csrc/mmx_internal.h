// mmx_internal.h -- data structures shared by the translation units of libmmx (not part of
// the ABI).  Notation follows the paper: m (reduced magnetisation), Ms, A, alpha, B_eff,
// tau, u (displacement), v (velocity), eps (strain).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/mmx.h"

#define MMX_MAX_STAGES 8
#define MMX_MATW 32  // floats per (sublattice, region) row of the device material table
#define MMX_HIST 4096

// indices into a device material row
enum {
  MP_MS = 0, MP_INVMS, MP_A, MP_D, MP_ALPHA, MP_LLG /* gamma/(1+alpha^2) */,
  MP_KU2 /* 2Ku1/Ms */, MP_UX, MP_UY, MP_UZ,
  MP_KC2 /* 2Kc1/Ms */, MP_C1X, MP_C1Y, MP_C1Z, MP_C2X, MP_C2Y, MP_C2Z, MP_C3X, MP_C3Y, MP_C3Z,
  MP_MEL1 /* 2B1/Ms */, MP_MEL2 /* 2B2/Ms */, MP_B1, MP_B2,
  MP_ZLB /* mu_B pol / (e Ms (1+xi^2)) */, MP_XI, MP_POL,
  MP_COUNT
};

// Device-resident step controller.  One instance per world.
struct MmxCtrl {
  double t, dt, tol;
  double err_last, max_torque;
  double t_end, torque_stop, dt_max;
  long long accepted, rejected, attempts, target_accepted;
  int sel;       // which of the two state buffers holds the accepted state
  int active;    // 0: all kernels of further attempts are no-ops
  int fixed;     // 1: accept unconditionally, keep dt
  int nan_flag;
  int order;     // order used by the step-size rule
  int hist_n;    // number of entries ever written to hist (ring buffer)
  unsigned err_bits, tq_bits;           // float bit patterns, atomicMax targets
  float ca[MMX_MAX_STAGES][MMX_MAX_STAGES];  // dt * a[i][j]; row s = b (non-FSAL final)
  float ce[MMX_MAX_STAGES];                  // dt * e[j]
  float cc[MMX_MAX_STAGES];                  // c[i] (stage times)
  double hist[MMX_HIST];
};

struct MmxTableau {
  int stages;
  int fsal;
  int order;      // convergence order (Table 2)
  int embedded;   // has an error estimate
  double c[MMX_MAX_STAGES];
  double a[MMX_MAX_STAGES][MMX_MAX_STAGES];
  double b[MMX_MAX_STAGES];
  double e[MMX_MAX_STAGES];
};

// Parameters of the fused local-field / torque / RK-combine kernel (local.cu).
struct LocalArgs {
  int nx, ny, nz, S, nreg;
  int per[3];
  float inv_h[3], inv_h2[3];
  const uint16_t* reg;   // null when nreg == 1
  const float* mat;      // [S][nreg][MMX_MATW]
  float scaleA11, scaleA12, A12, a0pref, Dinter;
  float dhomo[3];        // DMI vector of Eq.6, J/m^3
  float dmiq[4][3][3];   // general DMI tensor of Eq.4 as per-axis vectors q_i: sublattice 0, 1, 2, inter-sublattice; J/m^2
  int has_dmiq;          // any tensor set (routes the world to the general kernel)
  int has_dmiq12;        // the inter-sublattice one
  // Slonczewski torque (reading S37)
  int has_sl;
  float sl_beta;         // hbar jz / (e d): times 1/Ms gives beta in tesla
  float sl_mp[3], sl_l2, sl_epsp;
  float bext[3], J[3];
  unsigned terms;
  int has_J;
  int relax;             // 1: damping-only torque (mmx_relax, reading S39)
  int neumann;           // 1: Neumann boundary condition of Eq.5 (ghost cells, reading S41); 0: open (S9)
  // inputs.  A "sel pair" p[2] is indexed with ctrl->sel inside the kernel.
  const float* yin[2];     // stage state [nvec][3][N]
  const float* bdemag;     // [3][N] or null
  const float* strain;     // [6][N] or null
  // outputs
  float* kout[2];          // torque of this stage [nvec][3][N]
  float* heff_out;         // when non-null: write B_eff of sublattice heff_s here, nothing else
  int heff_s;
  float* tau_out;          // when non-null: write tau of sublattice heff_s here, nothing else
  // RK epilogue
  int stage;               // index i of k_i being computed (0-based)
  int n_prev;              // number of earlier k_j that enter the combination
  const float* kprev[2][MMX_MAX_STAGES];
  const float* y0[2];
  float* ynext[2];         // null: no combine
  int combine_row;         // row of ctrl->ca used for ynext
  int do_err;              // accumulate the embedded error norm
  int do_tq;               // accumulate max |k|
  MmxCtrl* ctrl;
  size_t vec_stride;       // 3*N
};

struct ElasticArgs {
  int nx, ny, nz, S, nreg;
  int per[3];
  float inv_h[3];
  const uint16_t* reg;
  const float* mat;
  float C11, C12, C44, inv_rho;
  int face;        // traction face or -1
  float tvec[3];
  double tamp, tfreq;
  const float* yin[2];
  float* strain;   // [6][N]  eps(u): magnetoelastic field, strain energy
  float* strain_f; // [6][N]  eps(u) + beta eps(v): stress of the elastic force when beta != 0, else null
  float beta;      // Rayleigh stiffness coefficient, s
  float* kout[2];
  float* accel_out;  // non-null: write the acceleration only
  int stage, n_prev;
  const float* kprev[2][MMX_MAX_STAGES];
  const float* y0[2];
  float* ynext[2];
  int combine_row;
  MmxCtrl* ctrl;
  size_t vec_stride;
  double t_fixed;   // used when ctrl == null (eval calls)
};

struct DemagPlan {
  int nx, ny, nz;
  int px, py, pz;      // transform lengths (1 = axis not transformed)
  int xc, xp;          // px/2+1 kept columns, padded row pitch (complex elements)
  int ky, kz;          // kernel octant extents along y, z (py/2+1 or 1)
  float2* tw[3];       // twiddle tables per axis
  float2* spec1;       // [3][nz][ny][xp]
  float2* spec2;       // [3][nz][py][xp]  (3-D only)
  float* khat;         // [6][kz][ky][xp]
  bool tiled;          // 3-D fast path: spec2 is tile-major and the kernel spectrum is stored as images (demag_tile.cu)
  float* kimg;         // [(py/2+1) ntx + py/16][6][65][16] (tiled only; khat is then not kept on the device)
  bool ready;
};

// kernel categories of the built-in profiler (mmx_profile_*)
enum { PK_X_FWD = 0, PK_MID_FWD, PK_INNER, PK_MID_INV, PK_X_INV, PK_LOCAL, PK_COMBINE, PK_CTRL, PK_STRAIN,
       PK_ELASTIC, PK_ENERGY, PK_COUNT };

struct ProfRec {
  int cat;
  cudaEvent_t e0, e1;
};

// a tensor map (CUtensorMap, 128 bytes) of one state buffer, for the TMA halo tiles of local.cu
struct MmxTmap {
  alignas(64) unsigned char bytes[128];
  const float* base;
};

struct mmx_world {
  int grid[3];
  double cell[3];
  int pbc[3];
  int S;
  int nvec;            // S (+2 with elastic)
  size_t N;
  cudaStream_t stream;
  bool own_stream;     // created by the library because the caller passed the legacy default stream
  int sm_count;        // multiprocessors of the device (grid size of the persistent kernels)
  int nreg;
  uint16_t* d_reg;
  std::vector<mmx_material> mats;  // [S][nreg]
  float* d_mat;
  bool mat_dirty;
  mmx_coupling cpl;
  double bext[3], J[3];
  double dmiq[4][9];   // general DMI tensors (mmx_set_dmi_tensor): sublattice 0, 1, 2, inter-sublattice; zero = none
  bool has_dmiq;
  mmx_slonczewski sl;  // jz = 0: off
  int boundary;        // MMX_BC_OPEN / MMX_BC_NEUMANN (non-periodic axes)
  bool relax_mode;     // stepping inside mmx_relax: the local kernels drop the precession term
  bool has_elastic;
  mmx_elastic el;
  bool use_demag;
  DemagPlan dm;
  // state and RK storage, each [nvec][3][N] floats
  float* Y[2];
  float* YS[2];
  float* K[MMX_MAX_STAGES + 1];
  float* bdemag;
  float* strain;
  float* strain_f;     // [6][N], only with viscous elastic damping
  float* scratch;      // [3][N]
  MmxCtrl* d_ctrl;
  unsigned* h_ctrl;    // mapped pinned host copy of the controller block's leading part (read_ctrl in api.cu)
  double* d_acc;       // fp64 accumulators for energies
  int sel_host;        // mirror of ctrl->sel valid when host_sel_valid
  bool k1_valid;       // FSAL k1 matches the current state
  int k1_method;
  long long dev_bytes;
  long long launches;
  bool prof;
  std::vector<ProfRec> prof_recs;
  // one attempt of an RK step captured as a CUDA graph (api.cu): every kernel argument of an attempt
  // is fixed between configuration changes (the "sel pairs" and the device-side controller were
  // designed for this), so a step is one graph launch instead of 27-39 kernel launches
  cudaGraphExec_t step_graph;
  int graph_method;
  long long graph_epoch, cfg_epoch;   // the graph is valid while graph_epoch == cfg_epoch
  long long graph_launches;           // kernels per replay
  bool use_graphs;
  MmxTmap tmaps[4];    // state buffers seen by the TMA local kernel (Y[0..1], YS[0..1]); reset by alloc_state
  int n_tmaps;
};

// RAII: brackets one kernel launch with CUDA events on the world's stream when profiling is on
struct ProfScope {
  mmx_world* w;
  ProfRec r;
  bool on;
  ProfScope(mmx_world* w_, int cat) : w(w_), on(w_->prof) {
    if (on) {
      r.cat = cat;
      cudaEventCreate(&r.e0);
      cudaEventCreate(&r.e1);
      cudaEventRecord(r.e0, w->stream);
    }
  }
  ~ProfScope() {
    if (on) {
      cudaEventRecord(r.e1, w->stream);
      w->prof_recs.push_back(r);
    }
  }
};

#ifdef __CUDACC__
// grid of a persistent kernel: every CTA resident from the start; CTAs per SM from the occupancy
// calculator, at most `want` per SM
template <typename K>
inline int mmx_persistent_grid(K kernel, int block, size_t smem, int sm_count, int want) {
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, block, smem) != cudaSuccess || per_sm < 1) {
    cudaGetLastError();
    per_sm = 1;
  }
  if (per_sm > want) per_sm = want;
  return per_sm * sm_count;
}

template <typename... KArgs, typename... Args>
inline cudaError_t mmx_launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args... args) {
  kernel<<<grid, block, smem, st>>>(KArgs(args)...);
  return cudaGetLastError();
}
#endif

// error plumbing (api.cu)
int mmx_fail(int code, const char* fmt, ...);
#define MMX_CUDA(call)                                                                   \
  do {                                                                                   \
    cudaError_t e__ = (call);                                                            \
    if (e__ != cudaSuccess)                                                              \
      return mmx_fail(MMX_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), \
                      __FILE__, __LINE__);                                               \
  } while (0)

// newell.cpp (host, fp64 / long double)
int mmx_newell_octant(const int grid[3], const double cell[3], const int pbc[3], double cutoff_cells,
                      std::vector<double>& out /* [6][n2][n1][n0] */, int n[3]);
int mmx_kernel_spectrum(const int grid[3], const int pbc[3], const int P[3], int xp,
                        const std::vector<double>& octant, const int n[3], double scale,
                        std::vector<float>& khat /* [6][kz][ky][xp] */);

// demag.cu
int mmx_demag_plan_sizes(mmx_world* w);
int mmx_demag_launch(mmx_world* w, const float* const yin[2], float* bout);

// demag_col.cu: register-resident column passes (fast path for P = 2 R^2 on a pruned axis)
struct InnerColLaunch {
  float2* spec;
  const float2* tw;
  int n_valid, p_outer, n_outer;
  size_t line_stride, comp_stride, outer_stride;
  size_t k_inner_stride, k_outer_stride, k_comp_stride;
  unsigned odd_inner, odd_outer;
};
bool mmx_inner_col_ok(const DemagPlan& d, int P, int n_valid);
int mmx_inner_col_launch(mmx_world* w, const InnerColLaunch& L);
bool mmx_mid_col_ok(int P, int n);
bool mmx_mid_pipe_ok(const mmx_world* w, int P, int nslab);

// demag_tile.cu: fused inner pass on the tile-major spectrum (3-D worlds with Pz = 128 on large grids)
bool mmx_tile_ok(const DemagPlan& d);
size_t mmx_tile_spec_elems(int py, int xc, int nz);
size_t mmx_tile_kimg_floats(int py, int xc);
void mmx_tile_kimg_build(const DemagPlan& d, const std::vector<float>& khat, std::vector<float>& out);
int mmx_inner_tile_launch(mmx_world* w);
int mmx_mid_col_launch(mmx_world* w, int P, int dir, const float2* in, float2* out, int n_in, int n_out,
                       size_t in_outer, size_t out_outer, int nslab, const float2* tw);

// demag_x.cu: warp-per-row-pair x passes (fast path for Px = 512, one region)
bool mmx_x_warp_ok(const mmx_world* w);
int mmx_x_warp_launch(mmx_world* w, int dir, const float* const yin[2], float* bout);

// local.cu
int mmx_local_launch(mmx_world* w, const LocalArgs& a);
int mmx_combine_launch(mmx_world* w, const float* const y0[2], const float* const k1[2],
                       float* const ynext[2], int row);
int mmx_controller_launch(mmx_world* w, const MmxTableau& tab, int mode);
int mmx_energy_launch(mmx_world* w, unsigned term_mask, const float* bdemag, double* host_out);

// stray.cu
int mmx_stray_launch(mmx_world* w, double height, double cutoff_cells, float* dev_out);

// elastic.cu
int mmx_strain_launch(mmx_world* w, const ElasticArgs& a);
int mmx_elastic_launch(mmx_world* w, const ElasticArgs& a);
int mmx_elastic_energy_launch(mmx_world* w, double* es, double* ek);
