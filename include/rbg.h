/*
 * rbg.h -- C ABI of the B200-native collision-term library (librbg.so).
 *
 * One thing is computed: the Monte Carlo evaluation of the relativistic 2->2 Boltzmann collision
 * term C_a[f](x,p1) at every phase-space cell -- Eq. 16 of arXiv 2308.04869
 * with the quantum factors of Eq. 18, summed over processes with the symmetry
 * factor of Eq. 19 -- and, optionally, the explicit collision update
 * f += dt*C of Eq. 27 with a count of cells that went negative.
 * The paper hands this integral to an external GPU Monte Carlo package; the
 * estimator, sampler and arithmetic order implemented here are fixed in DESIGN.md sections 2-4.
 *
 * Conventions
 *   - c = 1.  `hbar` (1 in the paper's own collision test) enters in two places: the occupation number
 *     nbar = (2 pi hbar)^3 f / g of Eq. 18 and the prefactor hbar^2 c |M|^2 / (64 pi^2 ...) of Eq. 16,
 *     i.e. C scales as hbar^2 for classical species.
 *   - All pointers named *_dev are DEVICE pointers (cudaMalloc / torch CUDA tensors); pointers
 *     named *_host are HOST pointers; everything else (structs, out-params) is host memory.
 *   - Layout of f, C, f_out: one contiguous array of doubles, species-major, then spatial cell,
 *     then momentum cell with pz fastest:
 *         index(s, ix, ipx, ipy, ipz) = off(s) + ix*Np(s) + (ipx*n_y(s) + ipy)*n_z(s) + ipz,
 *         off(s) = sum_{s'<s} Nx*Np(s'),   Np(s) = n_x(s) n_y(s) n_z(s),   Nx = nx*ny*nz,
 *     i.e. the paper's [nx,ny,nz,npx,npy,npz] array per species,
 *     concatenated over species.  Momentum cell centres: p_d = pmin_d + (i_d + 1/2) (pmax_d-pmin_d)/n_d.
 *   - Ownership: the caller owns every buffer it passes and must keep device buffers alive until
 *     the work queued on `cuda_stream` has completed.  The handle owns only its own scratch.
 *   - Calls that take a stream are asynchronous on that stream (a cudaStream_t passed as void*;
 *     NULL = the legacy default stream).  rbg_collision_host is synchronous.
 *   - Overlap: an output buffer must not share a byte with the f it is computed from (every kernel reads f at cells other
 *     than the one it writes); all entry points compare the byte ranges and return RBG_E_INVALID_ARG on any overlap.
 *   - Errors: every int-returning entry point returns RBG_OK (0) or a negative RBG_E_* code; the
 *     text is available from rbg_last_error().  No exception crosses this boundary.  There is no
 *     CPU fallback: anything the CUDA path does not support is an error, never a slow path.
 *   - Determinism: the result of rbg_collision / _update / _evolve / _host is a pure function of (f, the rbg_create
 *     arguments, n_samples, seed), bit for bit: it does not depend on the stream, on any rbg_set_option knob (CTA
 *     size, tile size, samples per lane, gather path) or on how spatial cells are partitioned across calls or GPUs
 *     (the sample stream is keyed by the global cell index; lane l of the warp that owns a momentum cell adds its samples
 *     n = l, l + 32, l + 64, ... in ascending order into ONE accumulator, whatever the samples-per-lane setting, and the 32
 *     lane sums are then combined by a fixed xor-shuffle tree: offsets 16, 8, 4, 2, 1).  rbg_collision_symmetric uses
 *     atomics: reproducible to rounding only.
 */
#ifndef RBG_H_
#define RBG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RBG_OK             0
#define RBG_E_INVALID_ARG (-1)
#define RBG_E_UNSUPPORTED (-2)
#define RBG_E_CUDA        (-3)

/* rbg_create flags */
#define RBG_FP64            0   /* sampling, kinematics and accumulation in fp64 (configs 1-4)        */
#define RBG_FP32_KINEMATICS 1   /* fp32 sampling + kinematics, fp64 accumulation (config 5)           */

typedef struct rbg_handle rbg_handle;   /* opaque; created by rbg_create, freed by rbg_destroy */

/* Only the number of spatial cells matters: Eq. 16 is local in x (all four distributions are taken
 * at the same (t,x)).  ix_offset is added to the local cell index when keying
 * the sample stream, so that a shard holding cells [ix_offset, ix_offset+nx*ny*nz) of a larger
 * domain reproduces the single-GPU result. */
typedef struct { int nx, ny, nz; int ix_offset; } rbg_spatial_grid;

/* Uniform, cell-centred Cartesian momentum grid of one species. */
typedef struct { int n[3]; double pmin[3]; double pmax[3]; } rbg_momentum_grid;

/* stat: 0 Boltzmann, +1 Bose-Einstein, -1 Fermi-Dirac (theta of Eq. 18); g: degrees of freedom
 * (Eq. 18: electrons 2, photons 1, quarks 6, gluons 16).  charge is carried for completeness; the
 * collision term does not use it. */
typedef struct { double mass; double charge; int stat; double g; } rbg_species;

typedef enum {
    RBG_M2_CONST            = 0,  /* |M|^2 = par[0]                                   */
    RBG_M2_COULOMB_SCREENED = 1,  /* |M|^2 = par[0] / (t - par[1]^2)^2                */
    RBG_M2_TCHAN_S2         = 2,  /* |M|^2 = par[0]^4 s^2 / (t - par[1]^2)^2   (Table III t-channel
                                     form with regulator)          */
    RBG_M2_ISO_DSIGMA       = 3,  /* |M|^2 = 64 pi^2 s par[0]: a constant differential cross section
                                     dsigma/dOmega = par[0], isotropic in the CM frame -- how the paper's
                                     collision test quotes its processes (Eq. 48, PAPER.md:493-500;
                                     cross section <-> matrix element Eq. 20-22, PAPER.md:214-230;
                                     DESIGN.md reading R17)                           */
    /* Table III of the paper: |M|^2 of the 2->2 parton processes of QCD, summed over the helicities
     * and colours of all four particles; par[0] = g, par[1] = m_g (the regulator m_g^2 is subtracted from t and u in
     * the denominators); SU_c(3): d_F = C_A = 3, C_F = 4/3, d_A = 8.  t = (k1 - k3)^2, u = (k1 - p)^2 of the process as
     * written a(k1) + b(k2) -> c(k3) + d(p).  With A = 8 g^4 d_F^2 C_F^2 / d_A, B = 16 g^4 d_F C_F (C_F - C_A/2),
     * C = 8 g^4 d_F C_F^2, D = 8 g^4 d_F C_F C_A, T = t - m_g^2, U = u - m_g^2:                                        */
    RBG_M2_QCD_Q1Q2         = 4,  /* q1 q2 -> q1 q2 (any mix of q, qbar of two flavours): A (s^2+u^2)/T^2                */
    RBG_M2_QCD_Q1Q1         = 5,  /* q1 q1 -> q1 q1: A [(s^2+u^2)/T^2 + (s^2+t^2)/U^2] + B s^2/(T U)                      */
    RBG_M2_QCD_Q1QB1        = 6,  /* q1 qbar1 -> q1 qbar1: A [(s^2+u^2)/T^2 + (u^2+t^2)/s^2] + B u^2/(T s)                */
    RBG_M2_QCD_Q1QB1_Q2QB2  = 7,  /* q1 qbar1 -> q2 qbar2: A (t^2+u^2)/s^2                                               */
    RBG_M2_QCD_QQB_GG       = 8,  /* q1 qbar1 -> g g: C (u/T + t/U) - D (t^2+u^2)/s^2                                     */
    RBG_M2_QCD_QG           = 9,  /* q1 g -> q1 g: D (s^2+u^2)/T^2 - C (u/s + s/U)                                        */
    RBG_M2_QCD_GG           = 10  /* g g -> g g: 16 g^4 d_A C_A^2 (3 - s u/T^2 - s t/U^2 - t u/s^2)                       */
} rbg_m2_kind;

/* How the CM scattering direction of a process is drawn (both estimate the same integral):
 *   RBG_SAMPLER_UNIFORM   uniform on the sphere;
 *   RBG_SAMPLER_TCHANNEL  polar angle about the CM direction of the grid particle drawn from the shape
 *                         1/(t - par[1]^2)^2 of the screened t-channel kinds by its inverse CDF, azimuth
 *                         uniform; the angular factor of |M|^2 then cancels in the weight (DESIGN.md
 *                         section 4b).  Only for elastic processes of RBG_M2_COULOMB_SCREENED / RBG_M2_TCHAN_S2 with par[1] != 0;
 *                         removes the (p* / par[1])^2-sized variance of sampling a forward peak uniformly. */
#define RBG_SAMPLER_UNIFORM  0
#define RBG_SAMPLER_TCHANNEL 1

/* Process a + b -> c + d (species indices), Eq. 16.  It contributes to the collision term of every
 * external species ("roles"): seen from a and from b, and, when it is inelastic ({c,d} != {a,b}),
 * through the reverse reaction (same |M|^2, "M_{ab<->cd}") also from c and from d.  An elastic process is written
 * c == a, d == b (a + b -> b + a is refused: t and u would be ambiguous).
 * sym < 0 selects the paper's rule ("1/2 ... when all incident particles are of the same type"): per
 * role, 1/2 if the two particles of the pair opposite the grid particle's pair are of one species, else 1; for an
 * elastic process that is 1/2 iff a == b.  sym >= 0 is used for every role of the process.
 * Degrees of freedom (reading R21): f is summed over the g internal states of its species.
 * Kinds 0..3 give |M|^2 of a + b -> c + d averaged over the states of a and b and summed over those of c and d; the
 * reverse direction is rescaled by g_a g_b / (g_c g_d).  The Table III kinds are summed over all four.  For elastic
 * processes of kinds 0..3 no factor appears. */
typedef struct { int a, b, c, d; int kind; double par[4]; double sym; int sampler; } rbg_process;

/* Create a handle.  Returns RBG_OK and stores the handle in *out, or a negative code (then *out
 * is NULL and rbg_last_error(NULL) has the text).  Rejects: non-positive grid counts,
 * pmax <= pmin, negative mass, stat not in {0,+1,-1}, g <= 0, species index out of range,
 * unknown kind, sampler or flags, a sampler that does not fit the kind or an inelastic process, a process
 * written a + b -> b + a, no CUDA device.  RBG_E_UNSUPPORTED: a species that takes part in a process has a momentum
 * cell centre of (numerically) zero energy, sqrt(|p|^2 + m^2) <= 1e-6 of the smallest cell width -- a massless species
 * on an odd grid symmetric about 0: Eq. 16 carries 1/p^0 of the grid particle, which diverges there. */
int rbg_create(rbg_handle** out, const rbg_spatial_grid* grid, int n_species, const rbg_species* species,
               const rbg_momentum_grid* momentum_grids /* [n_species] */, int n_process,
               const rbg_process* processes, double hbar, int flags);

/* C_dev[all cells] = collision term of f_dev (C_dev is overwritten, not accumulated into).
 * n_samples Monte Carlo samples per (role, spatial cell, momentum cell); seed keys the Philox
 * streams.  f_dev and C_dev hold rbg_f_elems() doubles and must not overlap. */
int rbg_collision(rbg_handle* h, const double* f_dev, double* C_dev, int n_samples, uint64_t seed,
                  void* cuda_stream);

/* Fused explicit Euler step: f_out_dev = f_dev + dt * C[f_dev].  `dt` is the EFFECTIVE step: Eq. 27 of the paper's
 * splitting reads (1/3) df/dt = C, so a caller reproducing it passes 3 * (the time step), as
 * rbg_be_step does; the same holds for rbg_collision_evolve.  *neg_flag_dev (one int in device memory, zeroed by the
 * caller) is incremented by the number of cells with f_out < 0; f_out is stored unclamped (policy is the caller's).
 * f_out_dev must not overlap f_dev, not even partly (RBG_E_INVALID_ARG). */
int rbg_collision_update(rbg_handle* h, const double* f_dev, double* f_out_dev, double dt, int* neg_flag_dev,
                         int n_samples, uint64_t seed, void* cuda_stream);

/* n_steps explicit Euler steps in a row (the paper's collision test runs 25 000 of them,
 * PAPER.md:504): f <- f + dt * C[f] with dt the effective step (see rbg_collision_update), step k (k = 0 .. n_steps-1) drawing its samples with seed + k, i.e.
 * exactly n_steps calls of rbg_collision_update ping-ponging between f_dev and scratch_dev (rbg_f_elems()
 * doubles, caller-owned, must not overlap f_dev).  On return (stream order) f_dev holds the final state;
 * scratch_dev is clobbered.  *neg_flag_dev accumulates the negative cells of every step.  n_steps >= 0. */
int rbg_collision_evolve(rbg_handle* h, double* f_dev, double* scratch_dev, double dt, int n_steps,
                         int* neg_flag_dev, int n_samples, uint64_t seed, void* cuda_stream);

/* NEXT-3: this repo's conservative estimator of the same collision term.  PAPER.md:257 names "the symmetric sampling
 * method [57]" without defining it and Ref. [57] is not part of PAPER.md, so whether this is that method cannot be
 * checked; the reading implemented is DESIGN.md section 4c / R25.  Same samples as
 * rbg_collision, but the net rate of every sample is credited to all four particles of the sampled reaction -- + to the
 * cells of the grid particle and its partner, - to the cells of the other pair -- and C of a species is the average of
 * the equivalent estimators, so that what one cell gains another loses sample by sample: particle number is conserved
 * to rounding whenever no particle leaves the momentum box.  C_dev is overwritten.  fp64 only, uniform sampler only
 * (RBG_E_UNSUPPORTED otherwise).  The deposits are atomic adds, so the result is reproducible to rounding, not bitwise. */
int rbg_collision_symmetric(rbg_handle* h, const double* f_dev, double* C_dev, int n_samples, uint64_t seed,
                            void* cuda_stream);

/* Same as rbg_collision with HOST buffers: copies f_host to the device (handle-owned scratch),
 * runs the kernels, copies C back, synchronises.  Spatial cells are independent, so large problems are pipelined over
 * up to 16 chunks of cells on three handle-owned streams (copy-in of chunk k+1 and copy-out of chunk k-1 beside the
 * kernels of chunk k); the result is bit-identical to rbg_collision (the sample stream is keyed by the global cell).
 * Pinned host memory lets the copies overlap the kernels; pageable memory works but serialises them.  f_host and
 * C_host must not overlap. */
int rbg_collision_host(rbg_handle* h, const double* f_host, double* C_host, int n_samples, uint64_t seed);

/* The fused explicit update (rbg_collision_update, Eq. 27) with HOST buffers, pipelined over chunks of spatial
 * cells exactly like rbg_collision_host: f_out_host = f_host + dt C[f_host], bit-identical to the device entry point.
 * *neg_count_host (host int) is SET to the number of cells of f_out that are negative -- unlike the device
 * flag it does not accumulate across calls.  Synchronous; f_out_host must not overlap f_host. */
int rbg_collision_update_host(rbg_handle* h, const double* f_host, double* f_out_host, double dt, int* neg_count_host,
                              int n_samples, uint64_t seed);

/* ---- The steps either side of the collision term ---------------------------------
 * Moments of f per species and spatial cell (midpoint sums over the momentum grid, Int d3p -> Sum dp^3, c = 1):
 *   n = Int f, j^k = Int v^k f (Eq. 5-6), T^{mu nu} = Int d3p/p0 p^mu p^nu f (Eq. 9).
 * M_dev: [n_species][Nx][RBG_N_MOMENTS] doubles in the order n, jx, jy, jz, T00, T01, T02, T03, T11, T12, T13, T22,
 * T23, T33.  total_dev (may be NULL): [Nx][RBG_N_MOMENTS] = the sum over species (Eq. 7, 9).  em_dev (may be NULL):
 * [Nx][4] = (rho, Jx, Jy, Jz) = Sum_a Q_a (n_a, j_a) (Eq. 15).  All device pointers, caller-owned,
 * overwritten.  Asynchronous on cuda_stream. */
#define RBG_N_MOMENTS 14
int rbg_moments(rbg_handle* h, const double* f_dev, double* M_dev, double* total_dev, double* em_dev, void* cuda_stream);

/* The moments of ONE species without a handle and without a single device allocation by this library.
 *
 * Who this is for.  Everything else in this header goes through rbg_create, which calls cudaMalloc for its per-species
 * tables.  Some programs cannot do that at the point where they need the moments: a solver that has handed all of HBM to
 * its own pool at start-up (a further cudaMalloc then fails, or takes memory the pool believed it had), a time-step loop
 * that must not stall (cudaMalloc / cudaFree synchronise the whole device), or a plug-in running inside a host
 * application that forbids device allocations after initialisation.  Such a caller already owns f and a place for the
 * result; the only other memory the kernel needs is the species' 1/E_p table (8 bytes per momentum cell), and here that
 * table lives in a fixed array compiled into the library (`static __device__`, RBG_MOMENTS_STATIC_MAX_CELLS doubles =
 * 512 KB), which every GPU that loads librbg.so holds from module load until the process exits.
 *
 * What it computes.  The same 14 midpoint sums as rbg_moments for a species of mass `mass` on momentum grid `grid`
 * (Eq. 5-6 and 9): f_dev is [n_cells][n0*n1*n2] doubles (one species' block of the usual layout),
 * M_dev is [n_cells][RBG_N_MOMENTS] doubles in rbg_moments' order.  Both are device pointers on the CURRENT device,
 * caller-owned, M_dev overwritten.  Two launches on cuda_stream (fill the table, then reduce), asynchronous.  The table
 * holds the same bits as the one rbg_create builds, and the reduction is rbg_moments' unstaged kernel, so the result is
 * identical to rbg_moments where that call takes its unstaged kernel and agrees with its staged kernels to rounding
 * (a different summation order: within 1e-12 of the same sums over |f|).
 * No species totals and no (rho, J): with one species the caller has them already (Q n, Q j).
 *
 * Limits and errors.  grid->n[0]*n[1]*n[2] must not exceed RBG_MOMENTS_STATIC_MAX_CELLS: a larger grid is refused with
 * RBG_E_UNSUPPORTED and a message naming both numbers (it is never truncated).  Non-positive counts, pmax <= pmin,
 * negative mass, n_cells < 0 or null pointers give RBG_E_INVALID_ARG; n_cells == 0 is a no-op.  The text is read with
 * rbg_last_error(NULL).  The call makes no cudaMalloc, cudaFree, cudaMemcpy or other allocating runtime call.
 *
 * First call on a device.  The array's device address differs per GPU and is not known to host code until asked for, so
 * the first call made with a given device current looks it up (cudaGetSymbolAddress, which also makes the runtime load
 * this library's code onto that device if it has not yet) and remembers it for later calls.  Make that first call during
 * your own set-up, outside any stream capture.
 *
 * Sharing.  There is one array per GPU, shared by every call from every thread, and it keeps whatever the previous call
 * wrote.  Each call rewrites the cells it is about to read before it reads them, in stream order, so back-to-back calls on
 * ONE stream are safe whatever their grids.  Two calls that can run on the GPU at the same time (different streams, or
 * different host threads on different streams) race on the table unless species mass and grid are identical: order them
 * with an event, or keep this entry point on one stream. */
#define RBG_MOMENTS_STATIC_MAX_CELLS 65536
int rbg_moments_static(const rbg_momentum_grid* grid, double mass, int n_cells, const double* f_dev, double* M_dev,
                       void* cuda_stream);

/* One first-order UPFD (unconditionally positivity-preserving finite difference) step of the drift term, Eq. 25 with
 * Eq. 28-30, all three directions at once (reading R23):
 *   f_out(x) = [ f/3 + dt Sum_d |v_d| f(x - sign(v_d) dx_d e_d) / dx_d ] / [ 1/3 + dt Sum_d |v_d| / dx_d ],  v = p/E_p.
 * The spatial grid is the (nx, ny, nz) of rbg_create, ix = (i_x ny + i_y) nz + i_z.  bc[d]: 1 periodic, 0 wall; a wall
 * reflects with probability zeta in [0,1]: the value beyond it is zeta * f(wall cell, p_d -> -p_d),
 * which needs momentum grids symmetric about 0 when zeta != 0 (else RBG_E_UNSUPPORTED); zeta = 0 absorbs.
 * f_out_dev must not overlap f_dev, not even partly (RBG_E_INVALID_ARG).  Needs the whole spatial domain in this handle (ix_offset == 0): across GPUs the
 * stencil would need the paper's ghost-layer exchange, which is out of scope. */
typedef struct { double dt; double dx[3]; int bc[3]; double zeta; } rbg_drift_params;
int rbg_drift_step(rbg_handle* h, const double* f_dev, double* f_out_dev, const rbg_drift_params* p, void* cuda_stream);

/* One step of the second-order positivity-preserving flux-limited drift scheme, Eq. 31-33 (the first
 * printing of Eq. 33, theta = 1e-10; reading R26), periodic in x, y and z:
 *   f_out = f - 3 dt Sum_d (F_{i+1/2} - F_{i-1/2}) / dx_d.
 * Explicit: positive for 3 dt Sum_d |v_d| / dx_d <= 1/2.  Same buffers and restrictions as rbg_drift_step. */
int rbg_drift_step_pfl(rbg_handle* h, const double* f_dev, double* f_out_dev, double dt, const double* dx /* [3], host */,
                       void* cuda_stream);

/* One first-order UPFD step of the Vlasov term, Eq. 26 with Eq. 34, all three directions at once:
 *   f_out(p) = [ f/3 + dt Sum_d |F_d| f(p - sign(F_d) dp_d e_d) / dp_d ] / [ 1/3 + dt Sum_d |F_d| / dp_d ],
 * F = Q (E + v x B) with the species' charge and the fields of the spatial cell, E_dev and B_dev being
 * [Nx][3] doubles; periodic in every momentum direction.  f_out_dev must not overlap f_dev, not even partly (RBG_E_INVALID_ARG). */
int rbg_vlasov_step(rbg_handle* h, const double* f_dev, double* f_out_dev, double dt, const double* E_dev,
                    const double* B_dev, void* cuda_stream);

/* One time step dt of the Boltzmann equation by the paper's splitting, Eq. 25-27 ("solving the BE is
 * equivalent to solving above three equations"), in the order drift, Vlasov, collision (the paper does not state an
 * order; reading R24):
 *     f <- rbg_drift_step(f, dt)                       Eq. 25 / 30      (if do_drift)
 *     f <- rbg_vlasov_step(f, dt, E, B)                Eq. 26 / 34      (if do_vlasov; E_dev, B_dev as above)
 *     f <- f + 3 dt C[f]  (rbg_collision_update)       Eq. 27: (1/3) df/dt = C   (if do_collision; n_samples, seed;
 *                                                       do_collision == 2: C from rbg_collision_symmetric instead)
 * in place: on return (stream order) f_dev holds the new state; scratch_dev (rbg_f_elems() doubles, caller-owned, not
 * overlapping f_dev) is clobbered.  *neg_flag_dev accumulates the cells the collision update left negative (may be
 * NULL when do_collision == 0).  All launches go to cuda_stream back to back (capturable in a CUDA graph). */
typedef struct { double dt; double dx[3]; int bc[3]; double zeta; int n_samples; uint64_t seed;
                 int do_drift, do_vlasov, do_collision; } rbg_be_step_params;
int rbg_be_step(rbg_handle* h, double* f_dev, double* scratch_dev, const rbg_be_step_params* p, const double* E_dev,
                const double* B_dev, int* neg_flag_dev, void* cuda_stream);

/* Number of doubles in f / C / f_out. */
size_t rbg_f_elems(const rbg_handle* h);
/* Number of roles (a process seen from one grid species; a+b with a != b gives two). */
int rbg_n_roles(const rbg_handle* h);
/* Role r (0 <= r < rbg_n_roles) as rbg_create expanded it from the process list (Eq. 19; DESIGN.md
 * section 3): species[0..3] = the species of the grid particle 1, its sampled partner 2 and the other pair 3, 4;
 * *sym = the symmetry factor applied (1/2 iff species 3 == species 4, unless the process overrides it); *cl, *cg = the
 * degrees-of-freedom factors of the loss (1+2 -> 3+4) and gain (3+4 -> 1+2) directions (reading R21: 1 and 1 for an
 * elastic process of kinds 0..3); *process = index into the process list.  Roles are in process order; within a process:
 * seen from a, from b (if b != a), and for an inelastic process from c and from d (if d != c).  Out-parameters may be
 * NULL.  Host-only query (no CUDA work); RBG_E_INVALID_ARG for a bad handle or index. */
int rbg_role_info(const rbg_handle* h, int r, int species[4], double* sym, double* cl, double* cg, int* process);
/* roles * Nx * Np * n_samples summed over roles: the "collision samples" one sweep evaluates. */
uint64_t rbg_sample_evals(const rbg_handle* h, int n_samples);
/* Kernels launched by the most recent rbg_collision* call on this handle. */
int rbg_last_launch_count(const rbg_handle* h);
/* Launch geometry / kernel path knobs (0 = automatic).  Two groups of keys.
 * (i) Results do NOT depend on these, bit for bit (rbg_collision / _update / _evolve / _host):
 *   "warps_per_cta" (1..32), "p1_per_cta" (momentum cells per CTA, >= 1), "samples_per_lane" (1 or 2: samples a lane
 *   evaluates per loop iteration; CTAs of more than 12 warps -- 16 with RBG_FP32_KINEMATICS -- use 1), "gather" (1 shared
 *   memory, 2 global/L2).
 * (ii) These select a kernel with different arithmetic, so results agree with the other setting (and with the oracle) to
 *   rounding only, and are bit-identical only for a fixed setting:
 *   "moments_path" / "vlasov_path" (1: rbg_moments / rbg_vlasov_step use their general staged kernel even where the
 *   symmetric-grid kernel applies; the symmetric-grid kernels read a 1/E table of one octant, pair the cells at +p and -p
 *   before multiplying, and pre-scale the fields: moments within 1e-12 of the sums over |f|, a Vlasov step within 1e-14
 *   relative), "sym_tables" (1: rbg_collision_symmetric accumulates the deposits of a CTA in shared-memory tables and
 *   flushes them at its end, instead of one global atomic per deposit: another order of atomic additions).
 * Returns RBG_E_INVALID_ARG for an unknown key or value. */
int rbg_set_option(rbg_handle* h, const char* key, int value);
/* Text of the last error on this handle (or of the last failed rbg_create if h is NULL). */
const char* rbg_last_error(const rbg_handle* h);
void rbg_destroy(rbg_handle* h);

/* Measurement helper: runs a register-resident chain of independent FMAs on every SM and reports
 * the achieved rate.  what: 0 = fp64 FMA, 1 = fp32 FMA, 2 = int32 multiply-add (each re-using two of its three
 * operands), 3 = fp64 FMA naming three distinct register pairs per instruction (register-file read bandwidth, not
 * the FP64 lanes, limits it), 4 = the 32 x 32 -> 64-bit multiply of a Philox round.  *ops_per_s counts one FMA /
 * multiply as one operation.  Used by bench.py for the live roofline denominator and its context. */
int rbg_probe_alu_peak(int what, int iters, double* ops_per_s, void* cuda_stream);

/* Diagnostic of the CHECKED build (librbg_checked.so, `python -m paper_2308_04869_b200.build --checked`, -DRBG_CHECKED): the
 * kernels then verify every index into a shared-memory or global table, the shared-memory layout of every CTA and, in the
 * persistent moments / Vlasov kernels, that a ring slot still holds the unit a warp believes it is consuming when it starts
 * and when it finishes reading it.  counts[0..7] receive the failures seen since the library was loaded, by class: f-table
 * index, tile index, direction-table index, output index, shared-memory layout, ring-slot contents, stencil / moment
 * index, conservative-estimator index; all must be 0.  Synchronises the device.  In the normal build the checks are
 * compiled out and the call returns RBG_E_UNSUPPORTED with all counts 0. */
#define RBG_SELFCHECK_CLASSES 8
int rbg_selfcheck_failures(uint64_t* counts /* [RBG_SELFCHECK_CLASSES], host */);

/* Diagnostic: compares the kernels' own fp64 and fp32 divide / reciprocal / square-root sequences
 * (the round-to-nearest fast paths without range checks) bit for bit with the
 * CUDA library operators on n_operands random operand sets (10 comparisons each); *mismatches must
 * come back 0.  Synchronous, default stream. */
int rbg_selftest_math(uint64_t n_operands, uint32_t seed, uint64_t* mismatches);

#ifdef __cplusplus
}
#endif
#endif /* RBG_H_ */
