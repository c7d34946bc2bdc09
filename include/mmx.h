/* mmx.h -- C-ABI boundary of the B200-native micromagnetic hot path.
 *
 * The calls follow the statement of the problem in arxiv 2411.18194 (mumax+),
 * cited as P:L<line> of PAPER.md: a simulation *world* holds one magnet
 * with 1 or 2 sublattices; the magnet has per-region
 * material parameters; the effective field (Eq.3, Eq.4, Eq.9, P:L116,
 * P:L142-144) enters the LLG torque (Eq.2) which is advanced in
 * time by an explicit / embedded Runge-Kutta method (Table 2),
 * optionally together with the elastodynamic equation (Eq.7-8).
 *
 * Conventions
 *   - plain C, no C++/torch types; every call returns an mmx_status (0 = OK),
 *     never throws, never aborts.  mmx_last_error() gives the message of the
 *     last failing call on this thread.
 *   - units are SI: lengths m, fields T, Ms A/m, A J/m, K J/m^3, D J/m^2,
 *     torque 1/s, current density A/m^2, time s.
 *   - vector fields are fp32, structure-of-arrays [3][Nz][Ny][Nx], x fastest.
 *   - pointers are tagged MMX_HOST or MMX_DEVICE by an explicit `mem` argument;
 *     the caller owns every pointer it passes, the library never keeps it
 *     after the call returns.  The world owns all of its device storage.
 *   - all device work is enqueued on the CUDA stream given at creation
 *     (NULL: the library creates its own blocking stream, see mmx_world_create).
 *     Calls with host out-parameters and the stepping calls synchronise that
 *     stream; the others are asynchronous.
 *   - there is no CPU fallback: without a CUDA device mmx_world_create fails
 *     with MMX_ECUDA.
 */
#ifndef MMX_H
#define MMX_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mmx_world mmx_world; /* opaque, library-owned */

typedef enum {
  MMX_OK = 0,
  MMX_EINVAL = -1, /* bad argument (NULL, size, non power-of-two periodic axis ...) */
  MMX_ENOMEM = -2, /* host or device allocation failed */
  MMX_ECUDA = -3,  /* a CUDA runtime call or kernel failed; no device */
  MMX_ESTATE = -4, /* call order (e.g. demag term requested before mmx_demag_kernel_init) */
  MMX_ENAN = -5    /* NaN/Inf reached the error or torque reduction */
} mmx_status;

enum { MMX_HOST = 0, MMX_DEVICE = 1 };

/* effective-field term bits for term_mask arguments */
enum {
  MMX_T_EXCH = 1,        /* Eq.3 first term: 2 A11/Ms lap m */
  MMX_T_DMI = 2,         /* Eq.4 interfacial subset, same sublattice */
  MMX_T_ANIS_U = 4,      /* uniaxial Ku1 */
  MMX_T_ANIS_C = 8,      /* cubic Kc1     */
  MMX_T_ZEEMAN = 16,     /* external field     */
  MMX_T_DEMAG = 32,      /* magnetostatic field */
  MMX_T_A12 = 64,        /* Eq.3 second term: A12/Ms lap m'                            */
  MMX_T_A0 = 128,        /* Eq.3 third term: 4 A0/(a^2 Ms) m'                          */
  MMX_T_DMI_INTER = 256, /* Eq.4 with the inter-sublattice tensor                      */
  MMX_T_MEL = 512,       /* Eq.9 magnetoelastic field */
  MMX_T_DMI_HOMO = 1024, /* Eq.6 homogeneous DMI between the sublattices */
  MMX_T_ALL = 2047
};

/* state fields for mmx_set_state / mmx_get_state */
enum { MMX_F_M0 = 0, MMX_F_M1 = 1, MMX_F_U = 2, MMX_F_V = 3, MMX_F_M2 = 4 /* third sublattice */ };

/* Runge-Kutta methods (Table 2; RK4 = classical, not in the table) */
enum {
  MMX_RK4 = 0,      /* classical 4th order, fixed step only            */
  MMX_DP45 = 1,     /* Dormand-Prince 5(4), FSAL   (Table 2 row 5)     */
  MMX_HEUN12 = 2,   /* Heun 2(1)                   (Table 2 row 1)     */
  MMX_BS23 = 3,     /* Bogacki-Shampine 3(2), FSAL (Table 2 row 2)     */
  MMX_CK45 = 4,     /* Cash-Karp 5(4)              (Table 2 row 3)     */
  MMX_RKF45 = 5     /* Fehlberg 5(4)               (Table 2 row 4)     */
};

/* Per (sublattice, region) material parameters ("material parameters"). */
typedef struct mmx_material {
  double Ms;      /* saturation magnetisation, A/m; 0 = empty cell                     */
  double A;       /* exchange stiffness A11, J/m                                       */
  double alpha;   /* Gilbert damping                                                   */
  double Ku1;     /* uniaxial anisotropy constant, J/m^3                               */
  double Kc1;     /* cubic anisotropy constant, J/m^3                                  */
  double D;       /* interfacial DMI strength of this sublattice, J/m^2                */
  double B1, B2;  /* magnetoelastic coupling constants, J/m^3 (Eq.8-9)                 */
  double pol;     /* spin polarisation of the current (Zhang-Li)                       */
  double xi;      /* non-adiabaticity (Zhang-Li)                                       */
  double gamma;   /* gyromagnetic ratio, rad/(T s); <= 0 selects 1.7595e11             */
  double u[3];    /* uniaxial axis (unit vector)                                       */
  double c1[3];   /* cubic axes c1, c2 (unit, orthogonal); c3 = c1 x c2                */
  double c2[3];
} mmx_material;

/* Inter-sublattice coupling and grain-boundary scaling (Eq.3). */
typedef struct mmx_coupling {
  double A0;        /* homogeneous inter-sublattice exchange, J/m                      */
  double A12;       /* inhomogeneous inter-sublattice exchange, J/m                    */
  double latcon;    /* lattice constant a of Eq.3, m                                   */
  double D_inter;   /* inter-sublattice interfacial DMI, J/m^2                         */
  double scale_A11; /* factor on A11 between cells of different regions (1 = none)     */
  double scale_A12; /* factor on A12 between cells of different regions                */
  double d_homo[3]; /* DMI vector d of Eq.6, J/m^3: energy density d . (m1 x m2), m1 / m2 the  */
                    /* first / second sublattice (the paper does not fix the order: a reading) */
} mmx_coupling;

/* Elastic medium (Eq.7) and one optional time-harmonic traction. */
typedef struct mmx_elastic {
  double C11, C12, C44;   /* cubic stiffness constants, Pa                             */
  double rho;             /* mass density, kg/m^3                                      */
  int traction_face;      /* -1 none; 0:x- 1:x+ 2:y- 3:y+ 4:z- 5:z+                    */
  double traction_vec[3]; /* direction of t in sigma.n = t                             */
  double traction_amp;    /* Pa                                                        */
  double traction_freq;   /* Hz; t(t) = amp * sin(2 pi freq t) * vec                   */
  double rayleigh_beta;   /* s; viscous term beta C : strain rate added to the stress  */
                          /* (Table 1 "stiffness coefficient of the Rayleigh   */
                          /* damping", 0.1 ps for NiO); 0 = undamped                   */
} mmx_elastic;

typedef struct mmx_rk_opts {
  int method;          /* MMX_DP45, ... (embedded pairs); MMX_RK4 only with fixed_dt    */
  int fixed_dt;        /* 1: every step accepted with dt = dt0 (parity / roofline runs) */
  double dt0;          /* first (or fixed) step; <= 0: 0.01 / max|torque| (adaptive)    */
  double tol;          /* accept iff err <= tol, err = dt*max_c |sum_j e_j k_j|_2       */
  long long nsteps;    /* stop after this many accepted steps (<= 0: no limit)          */
  double t_end;        /* stop when t >= t_end (<= 0: no limit)                         */
  double torque_stop;  /* stop when max|tau| < torque_stop [1/s] (<= 0: off)            */
  long long max_attempts; /* hard cap on attempted steps (<= 0: 1000000)                */
  double dt_max;       /* adaptive stepping never proposes a step above this (<= 0: none,  */
                       /* except with elastodynamics on, see mmx_step_rk45)              */
} mmx_rk_opts;

typedef struct mmx_rk_stats {
  long long accepted, rejected;
  double t;          /* simulation time after the call                                 */
  double dt;         /* step size proposed for the next step                           */
  double last_err;   /* error estimate of the last attempted step                      */
  double max_torque; /* max_c |tau_c| [1/s]: at the last accepted state for the FSAL     */
                     /* methods (DP45, BS23) and whenever the call stopped on            */
                     /* torque_stop; otherwise (RK4, Heun, CK45, RKF45) at the state     */
                     /* the last attempted step started from                             */
  long long launches;/* CUDA kernels launched by this call                             */
} mmx_rk_stats;

/* ---- life cycle ------------------------------------------------------------------- */

/* Message of the last failing call made by this thread ("" if none). */
const char* mmx_last_error(void);

/* Library version string. */
const char* mmx_version(void);
/* Layout revision of this header: raised whenever a struct that crosses the boundary changes size or field order, or an
 * enumerator changes value (3: mmx_rk_opts carries dt_max, 64 bytes; MMX_F_M2 = 4).  mmx_abi_version() returns the value the
 * library was built with; a caller compiled against another revision must not pass structs (compare once, at start-up). */
#define MMX_ABI_VERSION 3
int mmx_abi_version(void);

/* Create a world on the current CUDA device.
 *   grid[3]     = (Nx, Ny, Nz) cells, each >= 1
 *   cellsize[3] = (dx, dy, dz) in m
 *   pbc[3]      = number of periodic image repetitions per axis used by the demag kernel;
 *                 0 = open axis.  A periodic axis must have a power-of-two size.
 *   n_sublattices = 1 (ferromagnet), 2 (antiferro-/ferrimagnet) or 3 (non-collinear antiferromagnet: "a third
 *   sublattice with the same interaction terms as the first two": the inter-sublattice terms are summed over both partners,
 *   Eq.6 runs over the cyclic pairs (0,1), (1,2), (2,0); reading S38)
 *   cuda_stream = cudaStream_t (as void*) on which all work is enqueued.  NULL: the library
 *                 creates its own blocking stream (the legacy default stream cannot be captured
 *                 into the step graph); the runtime orders that stream against the legacy default
 *                 stream in both directions, so work the caller enqueues on stream 0 keeps its order.
 * Materials default to Ms = 0 everywhere until mmx_set_material is called. */
int mmx_world_create(const int grid[3], const double cellsize[3], const int pbc[3],
                     int n_sublattices, void* cuda_stream, mmx_world** out);
int mmx_world_destroy(mmx_world* w);

/* ---- parameters --------------------------------------------------------------------- */

/* Region index of every cell, [Nz][Ny][Nx] uint16 (P:L92 per-cell parameters, stored as a
 * region map + table).  n_regions >= 1; region_of_cell == NULL resets to one region. */
int mmx_set_regions(mmx_world* w, const uint16_t* region_of_cell, int mem, int n_regions);
/* Material of (sublattice, region); call after mmx_set_regions. */
int mmx_set_material(mmx_world* w, int sublattice, int region, const mmx_material* mat);
int mmx_set_coupling(mmx_world* w, const mmx_coupling* c);
int mmx_set_bext(mmx_world* w, const double B[3]);     /* uniform external (Zeeman) field, T */
int mmx_set_current(mmx_world* w, const double J[3]);  /* Zhang-Li current density, A/m^2 */
/* General intra-sublattice DMI of Eq.4: eps = sum_ijk D_ijk m_j d_i m_k, D_ijk = -D_ikj
 * (9 independent components).  q[3*i + l] is component l of the vector q_i of axis i, J/m^2, with
 * D_ijk = sum_l eps_jkl q_il, i.e. eps = sum_i q_i . (m x d_i m).  Uniform over the magnet; added to
 * the interfacial term of mmx_material.D under the same term bit MMX_T_DMI.  Interfacial D equals
 * q_x = D y^, q_y = -D x^; bulk DMI eps = D m.(curl m) equals q_i = -D e_i.  q = NULL clears it. */
int mmx_set_dmi_tensor(mmx_world* w, int sublattice, const double q[9]);
/* sublattice = MMX_DMI_INTER: the third tensor of Eq.4, "used to describe the intersublattice interaction",
 * D^(s,s') = D^(s',s): B^(s) = (2/Ms^(s)) sum_i q_i x d_i m^(s'), added to the interfacial mmx_coupling.D_inter
 * under the term bit MMX_T_DMI_INTER (two-sublattice worlds). */
#define MMX_DMI_INTER (-1)

/* Boundary condition on the non-periodic axes ("The Neumann boundary conditions as given in Eq. (5) are the
 * default in mumax+.  Alternatively, open or periodic boundary conditions can be used").
 *   MMX_BC_NEUMANN Eq.5, 2 A11 d_n m = A12 (d_n m' x m) x m + D.(n (x) m), as ghost cells (reading S41): the absent partner of
 *                  every exchange, A12 and DMI pair is m_c + h d_n m, with D.(n (x) m) = m x sum_i n_i q_i and the coupled
 *                  two-sublattice system solved in closed form.  The default of worlds with one or two sublattices, as in
 *                  the paper.  Without any DMI constant its solution is d_n m = 0 and the field equals the open one exactly.
 *   MMX_BC_OPEN    a stencil pair whose partner is absent (outside the grid, or Ms = 0) adds nothing (reading S9; the
 *                  natural boundary condition of the discrete pair energy).  The default of three-sublattice worlds (Eq.5
 *                  is written for a sublattice and its partner), opt-in otherwise; BASELINE.json's configurations ask for it
 *                  in words ("open boundaries").  With DMI it differs from Neumann by the h-independent local field
 *                  (1/(2 A Ms)) q_i x (m x q_i) on every boundary cell and every cell next to an empty one
 *                  (one sublattice): about half a tesla for D = 3 mJ/m^2, A = 15 pJ/m, Ms = 580 kA/m. */
enum { MMX_BC_OPEN = 0, MMX_BC_NEUMANN = 1 };
int mmx_set_boundary(mmx_world* w, int kind);

/* Slonczewski spin-transfer torque ("as formulated by ... Slonczewski [29], implemented in the same way
 * as in mumax3"; reading S37).  A current density jz through the free layer (thickness d), polarised along
 * the fixed-layer direction mp, adds in Gilbert form  gamma beta [eps m x (mp x m) - eps' m x mp],
 * beta = hbar jz/(e Ms d), eps = P L^2/((L^2 + 1) + (L^2 - 1) m.mp), P = mmx_material.pol; the explicit torque is
 * gamma beta/(1 + alpha^2) [(eps + alpha eps') m x (mp x m) - (eps' - alpha eps) m x mp].  NULL (or jz = 0) clears. */
typedef struct mmx_slonczewski {
  double jz;         /* current density through the layer, A/m^2                        */
  double mp[3];      /* fixed-layer polarisation direction (normalised by the library)  */
  double lambda;     /* Slonczewski Lambda (>= 1; 1: no angular dependence, eps = P/2)  */
  double eps_prime;  /* secondary (field-like) spin-torque parameter eps'               */
  double thickness;  /* free-layer thickness d, m; <= 0: Nz * cellsize[2]               */
} mmx_slonczewski;
int mmx_set_slonczewski(mmx_world* w, const mmx_slonczewski* s);
/* Enable elastodynamics (adds the fields U, V to the integrated state); NULL disables. */
int mmx_set_elastic(mmx_world* w, const mmx_elastic* e);
/* Switch the magnetostatic term on/off for stepping (default on once the kernel exists). */
int mmx_enable_demag(mmx_world* w, int on);

/* Copy a state field in / out: `field` = MMX_F_*; buf is fp32 [3][Nz][Ny][Nx] (the user's side of the state is
 * plain arrays).  m is taken as given: the caller passes unit vectors (or 0 in cells without a magnet). */
int mmx_set_state(mmx_world* w, int field, const float* buf, int mem);
int mmx_get_state(mmx_world* w, int field, float* buf, int mem);
int mmx_set_time(mmx_world* w, double t);
int mmx_get_time(mmx_world* w, double* t);

/* ---- magnetostatic kernel ---------------------------------------------------------------- */

/* Build the demagnetising tensor: Newell's analytic cell-cell tensor for
 * offsets closer than analytic_cutoff_cells * max(cellsize) (<= 0 selects 32), an
 * asymptotic (quadrature of the point-dipole tensor) form beyond; periodic images summed
 * on periodic axes.  The tensor is transformed (fp64, host), scaled by -mu0 / P and stored
 * as a real fp32 octant on the device.  One-time setup, not on the timed path. */
int mmx_demag_kernel_init(mmx_world* w, double analytic_cutoff_cells);

/* Host-only helper used by the tests: demag tensor N_ij (6 components xx,yy,zz,xy,xz,yz) on
 * the non-negative octant of offsets, fp64 [6][n2][n1][n0], for an open (pbc=0) or periodic
 * world.  n[a] = grid[a] on open axes, grid[a]/2+1 on periodic ones.  Needs no GPU. */
int mmx_newell_tensor_host(const int grid[3], const double cellsize[3], const int pbc[3],
                           double analytic_cutoff_cells, double* out, long long out_len);

/* Host-only helper used by the tests: the real kernel spectrum as stored on the device,
 * fp32 [6][KZ][KY][XP] with the factor -mu0/(Px Py Pz) folded in.  dims_out[5] receives
 * (Px, Py, Pz, XP, total element count); call with out == NULL to query the sizes. */
int mmx_kernel_spectrum_host(const int grid[3], const double cellsize[3], const int pbc[3],
                             double analytic_cutoff_cells, float* out, long long out_len,
                             long long dims_out[5]);

/* ---- evaluation ------------------------------------------------------------------------ */

/* Effective field of one sublattice, restricted to term_mask, of the current state (T).
 * out: fp32 [3][Nz][Ny][Nx].  Cells without a magnet (Ms = 0 for this sublattice) report 0 for every
 * term, the magnetostatic one included: B_eff is the field acting on m, the stray field in empty
 * cells is not part of this call.  mmx_eval_torque likewise reports 0 there. */
int mmx_eval_heff(mmx_world* w, int sublattice, unsigned term_mask, float* out, int mem);
/* Torque dm/dt (Eq.1-2 + Zhang-Li) of one sublattice for the current state (1/s), all
 * enabled terms. */
int mmx_eval_torque(mmx_world* w, int sublattice, float* out, int mem);
/* Elastic right-hand side: acceleration (f_el + sum_s f_mel)/rho  (Eq.7-8), m/s^2. */
int mmx_eval_accel(mmx_world* w, float* out, int mem);
/* Energy (J) of the terms in term_mask summed over sublattices, fp64 accumulation: -1/2 sum Ms V m.B for the terms
 * bilinear in m (the energy densities of Eq.4, and Eq.6, in their discrete pair form), -sum Ms V m.B for
 * the Zeeman term, -1/4 sum Ms V m.B for the quartic cubic anisotropy. */
int mmx_energy(mmx_world* w, unsigned term_mask, double* joule_out);
/* (1/2 sum sigma:eps V, 1/2 sum rho v^2 V) */
int mmx_elastic_energy(mmx_world* w, double* strain_energy, double* kinetic_energy);
/* max over cells and sublattices of |tau| (1/s): the measure of "relaxed". */
int mmx_max_torque(mmx_world* w, double* out);

/* Field of the magnet in a probe layer above it ("we calculate the out-of-plane component of the magnet's stray
 * field 60 nm above the film's surface", Fig.3; reading S40): the probe layer has the magnet's in-plane grid and
 * cell size, its cells are centred `height` metres above the top surface (height > -cellsize[2]/2), values are averages
 * over a probe cell.  B_i = -mu0 sum N_ij(x - x', y - y', Dz_k) M_j over all cells of all layers, M = sum_s Ms m_s, N the
 * Newell tensor at the real z offset Dz_k = (Nz - k - 1/2) dz + height.  Open boundaries only (MMX_EINVAL otherwise).
 * out: fp32 [3][Ny][Nx] tesla, host or device.  A direct sum: meant for imaging a state, not for the time loop. */
int mmx_stray_field(mmx_world* w, double height, float* out, int mem);

/* The same probe-layer field (Fig.3; P:L144 for M = sum_s Ms m_s; reading S40) for callers that may not allocate.
 *
 * mmx_stray_field cudaMallocs and cudaFrees its Newell table on every call and needs a world, which owns cudaMalloc'd
 * storage of its own.  Some callers cannot afford either: a process whose device memory is held in full by a pooling
 * allocator (PyTorch / CuPy caching allocator, a serving arena), where a raw cudaMalloc fails or forces the pool to be
 * flushed; a latency-bound loop, because cudaMalloc / cudaFree take a driver-wide lock and cudaFree waits for the device;
 * a thread that runs while another thread captures a CUDA graph in the global capture mode, which a cudaMalloc breaks.
 * mmx_stray_field_static is the entry point for them.  It needs no world.  It calls no cudaMalloc, cudaFree,
 * cudaMallocAsync or other allocating routine and uses no host heap; its only scratch memory, M = sum_s Ms m_s as
 * [3][Nz][Ny][Nx] fp32, lives in an array built into the library's CUDA module.
 *
 *   limit     Nx*Ny*Nz <= MMX_STRAY_STATIC_MAX_CELLS (262 144, e.g. 512 x 512 x 1; the paper's Fig.3 film is
 *             500 x 500 x 1).  Larger grids: MMX_EINVAL with a message that names the limit, nothing is launched.
 *   cost      12 * MMX_STRAY_STATIC_MAX_CELLS bytes = 3 MiB of device memory on every GPU on which the library's CUDA
 *             module gets loaded, from that moment until the process exits, whether or not this call is ever made.
 *   grid      (Nx, Ny, Nz), host.   n_sublattices 1..3.   Ms[n_sublattices] host, A/m, one value per sublattice (the
 *             magnet is uniform here: no region map; an empty cell is m = 0 in that cell).
 *   m         DEVICE, fp32 [n_sublattices][3][Nz][Ny][Nx], the reduced magnetisations.   Caller-owned, read only.
 *   table     DEVICE, fp32 [Nz][6][Ny][Nx]: the z-shifted Newell tensor per source layer with -mu0 folded in, exactly the
 *             numbers mmx_stray_table_host writes (build it once per grid / cell size / height, copy it into device
 *             memory you already own).  Caller-owned, read only.
 *   out       DEVICE, fp32 [3][Ny][Nx], tesla.  Caller-owned; every element is written.
 *   cuda_stream  cudaStream_t as void*; NULL = the legacy default stream.  Two kernels are enqueued on it and the call
 *             returns without waiting for them (read `out` in stream order, or after synchronising the stream).
 * All pointers must belong to the device that is current when the call is made.
 *
 * First call on a device.  The first call made with a given device current also does a one-time set-up for that device:
 * it asks the runtime for the device address of the built-in array (cudaGetSymbolAddress; this is also what makes the
 * runtime load the module there).  Make that first call -- one per device you use -- before any stream capture is started.
 *
 * Sharing.  Every call on a device uses the same array, and the array keeps what the previous call left in it.  Nothing
 * in it has to start at zero: a call overwrites elements [0, 3 Nx Ny Nz) before it reads them, in stream order.  Calls
 * that overlap in time on one GPU (different streams, several host threads, several worlds) race on the array and return
 * garbage without any error: order them on one stream, or with events.  Calls on different GPUs do not interact.
 *
 * Errors: MMX_EINVAL (NULL pointer, sizes, the limit above, a device ordinal >= 64), MMX_ECUDA (set-up or launch failed).
 * Pointers are not checked for being device pointers. */
#define MMX_STRAY_STATIC_MAX_CELLS 262144
int mmx_stray_field_static(const int grid[3], int n_sublattices, const double Ms[], const float* m, const float* table,
                           float* out, void* cuda_stream);
/* Host-only helper, needs no GPU: the table mmx_stray_field_static takes, fp32 [Nz][6][Ny][Nx] (components xx, yy, zz, xy,
 * xz, yz on the non-negative quadrant of in-plane offsets; layer k at z offset (Nz - k - 1/2) dz + height; times -mu0),
 * the same values mmx_stray_field builds internally.  out_len must be Nz*6*Ny*Nx.  Ordinary host code: it uses the host
 * heap and may take seconds on large grids; run it once, at set-up. */
int mmx_stray_table_host(const int grid[3], const double cellsize[3], double height, float* out, long long out_len);

/* ---- time stepping --------------------------------------------------------------------- */

/* nsteps classical RK4 steps of size dt (BASELINE config 1 protocol). */
int mmx_step_rk4(mmx_world* w, double dt, long long nsteps);
/* Embedded Runge-Kutta stepping (Table 2; default Dormand-Prince).  stats may be NULL.  The call
 * returns after the device has finished (it reads the controller block back).
 *   - t_end > 0 and the current time already >= t_end: nothing is done, MMX_OK, accepted = 0.
 *   - torque_stop: tested on the torque at the accepted state.  FSAL methods have it as the last
 *     stage of the step; the others (Heun, Cash-Karp, Fehlberg) evaluate it as the first stage of
 *     the next attempt and abandon that attempt (it counts neither as accepted nor as rejected).
 *   - the error estimate is taken over the magnetic variables only (the paper leaves adaptive
 *     stepping of the elastic variables to future work).  With elastodynamics on, adaptive
 *     stepping therefore clamps the step to dt_max, and dt_max <= 0 then selects the bound of the chosen method,
 *         dt_max = 0.9 y_max / omega_max,
 *     y_max = mmx_rk_imag_stability_limit(method, 1e-6), omega_max = 1.3722 v_max sqrt(sum_a 1/h_a^2) over the axes with
 *     more than one cell: 1.3722/h is the largest wave number the fourth-order first difference of Eq.7 can
 *     represent, v_max the fastest wave of the cubic medium (the largest of sqrt(C11/rho), sqrt(C44/rho) and the
 *     longitudinal velocities along [110] and [111]).  An undamped wave sits on the imaginary axis of the method's
 *     stability region; above y_max every step amplifies round-off, so a quiet magnet must not drive dt past it.
 *     Heun, Cash-Karp and Fehlberg are nowhere neutrally stable on that axis: their bound comes from the growth allowance
 *     (1e-6 per step) alone and is 2 to 20 times smaller than Dormand-Prince's.
 *   - MMX_ENAN: a NaN/Inf reached the error or torque reduction; the attempt is not accepted, the
 *     accepted state and time are left as they were, stepping stops. */
int mmx_step_rk45(mmx_world* w, const mmx_rk_opts* opts, mmx_rk_stats* stats);

/* Host-only helper, needs no GPU: how far up the imaginary axis a step of `method` (Table 2, or MMX_RK4) may
 * reach.  *y_max = the largest y with |R(i y')| <= 1 + growth for all 0 <= y' <= y, R the method's stability polynomial;
 * an undamped oscillation of angular frequency omega advanced with omega dt <= y_max is amplified by at most 1 + growth per
 * step.  growth = 0: RK4 2 sqrt 2, Bogacki-Shampine sqrt 3, Dormand-Prince 0.997, (almost) 0 for Heun, Cash-Karp, Fehlberg.
 * Resolution 1e-4, searched up to y = 4. */
int mmx_rk_imag_stability_limit(int method, double growth, double* y_max);

/* Relaxation ("after letting a non-collinear antiferromagnet relax from a random state"; DESIGN.md reading
 * S39): the precession term m x B of Eq.2 is dropped and the damping term -gamma alpha/(1+alpha^2) m x (m x B) is
 * integrated with adaptive Dormand-Prince steps (tolerance tol, <= 0: 1e-5) until max_c |tau_c| < torque_stop [1/s]
 * or max_attempts (<= 0: 1e6) attempts were made.  The simulation time is left where it was.  stats may be NULL. */
int mmx_relax(mmx_world* w, double torque_stop, double tol, long long max_attempts, mmx_rk_stats* stats);
/* Error estimates of the most recent attempted steps (newest last); returns the number
 * written through *n_out (at most n). */
int mmx_get_err_history(mmx_world* w, double* host_out, int n, int* n_out);

/* Built-in kernel timer: while enabled, every kernel launch is bracketed by CUDA events on the
 * world's stream.  mmx_profile_read synchronises, sums the elapsed milliseconds and launch counts
 * per kernel category into ms_out[n] / count_out[n] (n >= 11) and clears the records.
 * Categories: 0 demag x_fwd, 1 mid_fwd, 2 inner (fwd * K * inv), 3 mid_inv, 4 x_inv,
 * 5 local field/torque/RK, 6 RK combine, 7 controller, 8 strain, 9 elastic RHS, 10 energy. */
int mmx_profile_enable(mmx_world* w, int on);
int mmx_profile_read(mmx_world* w, double* ms_out, long long* count_out, int n);

/* Number of device bytes owned by the world. */
int mmx_device_bytes(mmx_world* w, long long* bytes);

/* CUDA-graph stepping.  mmx_step_rk4 / mmx_step_rk45 capture one attempt of a step (every kernel of
 * the step-size controller, the demag passes, the local and elastic kernels) as a CUDA graph on first
 * use and replay it per attempt; the graph is rebuilt after any mmx_set_* / mmx_enable_demag /
 * mmx_demag_kernel_init call and is bypassed while the profiler is on.  mmx_graph_enable(w, 0)
 * switches to plain launches (also: environment variable MMX_NO_GRAPH at world creation).
 * mmx_graph_info: *kernels_per_replay = kernels inside the instantiated graph, 0 if none is live. */
int mmx_graph_enable(mmx_world* w, int on);
int mmx_graph_info(mmx_world* w, long long* kernels_per_replay);

#ifdef __cplusplus
}
#endif
#endif /* MMX_H */
