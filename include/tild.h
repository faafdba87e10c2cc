/*
 * tild.h -- C-ABI of the B200-native TILD particle-mesh force path.
 *
 * The method is the per-time-step "Particle-to-Mesh" non-bonded force evaluation of
 * Theoretically-Informed Langevin Dynamics as described in PAPER.md (arxiv 2302.02474,
 * MATILDA.FT) section IV.C "Long-range interactions" (L221-231, Eq. 18, Fig. 1), applied to the
 * model of section III (Eq. 1-4; smearing L139-149), plus harmonic bonds (Eq. 2,
 * IV.B L207-209) and the GJF Langevin integrator (VI.B.6 L346-352).  The paper defines no API
 * (its user surface is an input script, L58-90); the arguments below follow its statement of the
 * model.  Readings of points where the paper is silent are listed in DESIGN.md ("A<n>").
 *
 * Conventions
 *  - Unless marked HOST, every pointer argument is a DEVICE pointer owned by the caller (e.g. a
 *    torch tensor's data_ptr).  The library never frees or reallocates caller memory.
 *  - `workspace` is caller-allocated device memory of at least tild_workspace_bytes() bytes,
 *    256-byte aligned, borrowed until tild_destroy().  The context owns only its cuFFT plans
 *    (and their work areas), CUDA events and host bookkeeping.
 *  - All calls enqueue on the `cuda_stream` given to tild_init (a cudaStream_t; NULL = legacy
 *    default stream) and return without synchronising, except where stated.
 *  - Layouts: positions/velocities/forces AoS [n][3] float (x[ind*Dim+j]);
 *    grids [species][Nx][Ny][Nz] float, z fastest, linear node index g = (ix*Ny + iy)*Nz + iz;
 *    force fields [species][3][Nx][Ny][Nz].  Box is [0,L) per axis, periodic, node g at g*h.
 *  - Return value: 0 on success, negative tild_status on failure; tild_last_error() gives text.
 *    No exceptions, no output to stdout/stderr, no environment variables.  The only process-wide state is the
 *    per-kernel shared-memory limit, which is only ever raised.  A context is bound to the CUDA device that was
 *    current at tild_init; its entry points switch to that device and back.
 *  - type[i] must be in [0, S) and bond_partner entries in [-1, n): tild_set_state checks both (synchronising once) and
 *    returns TILD_EINVAL; the stage calls trust their arguments.
 *  - There is no CPU fallback: every entry point that computes needs a CUDA device.
 */
#ifndef TILD_H
#define TILD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TILD_MAX_SPECIES 8
#define TILD_MAX_BONDS 4

typedef enum {
    TILD_OK = 0,
    TILD_EINVAL = -1,  /* bad sizes / order / non-positive box / struct_size mismatch / NULL */
    TILD_ENOMEM = -2,  /* workspace too small or misaligned */
    TILD_ECUDA = -3,   /* a CUDA runtime call failed */
    TILD_ECUFFT = -4,  /* a cuFFT call failed */
    TILD_ESTATE = -5   /* tild_step / tild_get_state before tild_set_state */
} tild_status;

/* flags */
#define TILD_FLAG_TIMING 1u        /* record CUDA events around every stage of tild_step */
#define TILD_FLAG_NAIVE_SPREAD 2u  /* per-particle global-atomic spread (baseline kernel) */
#define TILD_FLAG_NAIVE_INTERP 4u  /* per-particle global-gather interpolation (baseline kernel) */
#define TILD_FLAG_DECONVOLVE 16u   /* pair kernel u^(k) / W^(k)^2, W^ = prod_a sinc(k_a h_a/2)^P: undoes the smoothing of the
                                      order-P assignment (A13; default off: the kernel is exactly u^(k)) */
#define TILD_FLAG_SAMPLED_KERNEL 32u /* pair kernel = DFT of u_G sampled on the mesh (minimum image), as PAPER.md L223
                                      describes, instead of the analytic u^(k) (A5b); still three 1-D tables */
#define TILD_FLAG_PLAIN_FFT 64u    /* 3-D cuFFT plans + the element-wise k-space kernel even where the fused x-transform
                                      kernel applies (Nx in {16,32,64,128,256}, S <= 4).  For A/B runs: the results agree to fp32
                                      rounding */
#define TILD_FLAG_GRAPH 8u         /* accepted for compatibility: graph replay is the default (see TILD_FLAG_EAGER) */
#define TILD_FLAG_EAGER 256u       /* launch every kernel of every step individually.  Default: tild_step replays blocks of
                                      2*resort_every steps as one CUDA graph (launch-bound small systems: C1 0.066 -> 0.044 ms
                                      per step; a cycle that starts with the periodic return to particle-id order is a block of
                                      resort_every steps) whenever it can -- no TILD_FLAG_TIMING, an even resort_every, and a stream
                                      that can be captured (not the legacy default stream); otherwise it launches eagerly */
#define TILD_FLAG_2D 512u          /* two-dimensional system (Listing 1 L65; A27): grid[2] must be 1; the z
                                      coordinates are carried along unchanged, no force, noise or velocity along z.  box[2] is
                                      the thickness that turns the areal density into rho0 = n / V */
#define TILD_FLAG_EXTRAS 1024u     /* reserve workspace and plans for the extra mesh interactions: per-particle charges
                                      (tild_set_charges) and the Maier-Saupe interaction (mu_ms, tild_set_ms_partners) */
#define TILD_FLAG_NO_TMA 2048u     /* stage every tile image with cp.async, also where a TMA box applies (A/B runs) */
#define TILD_FLAG_HOST_PIPELINE 8192u /* workspace for tild_run_host_submit / _wait: device staging of one input and two output batches */
#define TILD_FLAG_ARRIVAL_SORT 16384u /* A/B: re-sorts hand out slots in arrival order (atomics) instead of keeping the order of the particles
                                        that stay in their segment */
#define TILD_FLAG_NO_DEFRAG 32768u  /* A/B: never put the state back into particle-id order (done every 5th re-sort for n >= 2^20 otherwise) */
#define TILD_FLAG_DEFRAG_SMALL 65536u /* ... also for smaller systems (tests) */
#define TILD_FLAG_GEN1_TILES 128u   /* first-generation tile kernels (32 bank classes with overflow rounds, per-particle work
                                      in class order) even where the rotation-class kernels apply (P = 4); for A/B runs */

/* integrators */
#define TILD_INTEGRATOR_GJF 0   /* Gronbech-Jensen & Farago, one force evaluation per step */
#define TILD_INTEGRATOR_EM 1    /* Euler-Maruyama: r' = r + (dt/gamma) F + sqrt(2 kT dt/gamma) xi; velocities unused */
#define TILD_INTEGRATOR_VV 2    /* velocity Verlet with the Langevin ExtraForce -gamma v + beta/dt in both half kicks, one noise
                                   per step (A24); gamma = 0: plain velocity Verlet;
                                   needs gamma dt / 2m < 1 */

typedef struct tild_ctx tild_ctx;

/* The model statement.  PAPER.md: box L54; grid Nx,Ny,Nz and pmeorder Listing 1 L69-78; species,
 * chi_ij, kappa Eq. 3-4; Gaussian range L121/L139-143; bonds Eq. 2; delt L71;
 * integrator L82/L352; reduced units (kT, m, b) L100. */
typedef struct {
    uint32_t struct_size;      /* = sizeof(tild_params) */
    int32_t n;                 /* particles, >= 0 */
    int32_t n_species;         /* S, 1..TILD_MAX_SPECIES */
    int32_t order;             /* P = grid nodes touched per dimension, 1..5 (A1: P = 2..5 are the paper's orders 1..4) */
    double box[3];             /* L > 0 */
    int32_t grid[3];           /* N >= P, each; any size cuFFT accepts (2,3,5,7 factors are fast) */
    int32_t max_bonds;         /* bond partner slots per particle, 0..TILD_MAX_BONDS */
    double chi[TILD_MAX_SPECIES * TILD_MAX_SPECIES]; /* chi[I*8+J], symmetric, diagonal ignored */
    double kappa;              /* Helfand compressibility, Eq. 4 */
    double a;                  /* smearing length of h(r), L139; used when sigma2 <= 0 */
    double sigma2;             /* variance of u_G (L121); <= 0 -> 2 a^2 (L143) */
    double rho0;               /* <= 0 -> n / V (L121) */
    double k_bond, r0_bond;    /* U_bond = k (|d| - r0)^2; Eq. 2 has k = 3/(2 b^2), r0 = 0 */
    double dt, gamma, kT, mass;/* GJF parameters (A11) */
    uint64_t seed;             /* Philox4x32-10 key (A12) */
    int32_t resort_every;      /* physically re-sort particles by cell every this many steps; <= 0 -> default */
    uint32_t flags;            /* TILD_FLAG_* */
    int32_t integrator;        /* TILD_INTEGRATOR_GJF (default, A11), TILD_INTEGRATOR_EM (overdamped, A11b; gamma > 0) or
                                  TILD_INTEGRATOR_VV (velocity Verlet + Langevin ExtraForce, A24) */
    int32_t tile_shape;        /* 0 = automatic: tiles of 8 x 16 x 32 cells, halved in y and then in z while there are fewer than
                                  296 tiles or more than 4096 particles per tile; else TY | TZ << 8 with TY in {8, 16}, TZ in {16, 32}
                                  (a zero byte leaves that edge automatic) */
    /* electrostatics on the same path (reading A22): valence per species, Bjerrum length
     * (0 = off), Gaussian smearing length of a charge; pair kernel 4 pi l_B exp(-k^2 a_q^2) / k^2, k = 0 dropped */
    double charge[TILD_MAX_SPECIES];
    double bjerrum;
    double a_charge;
    /* cosine (wormlike-chain) angle potential lambda [1 + cos(theta_ijk)], Eq. 16; 0 = none.  Needs
     * max_bonds == 2: the triplets are (partner slot 0, bead, partner slot 1) of every bead with both (A23) */
    double lambda_wlc;
    /* harmonic angle potential k_theta (theta_ijk - theta0)^2, Eq. 17, on the same triplets; k_theta = 0:
     * none; theta0 in [0, pi].  The force is singular at sin(theta) = 0 and that term is dropped there */
    double k_theta, theta0;
    /* Maier-Saupe parameter mu of PAPER.md Eq. 20 L241 (0 = off): beta U = -(mu/rho0) int int S(r) : S(r') u_G(|r - r'|) with the
     * orientation tensors S_i = u_i u_i - I/3 of the LC centres named by tild_set_ms_partners (A26) */
    double mu_ms;
} tild_params;

/* HOST. Bytes of device workspace tild_init needs for these parameters. */
int tild_workspace_bytes(const tild_params* params /*HOST*/, size_t* bytes /*HOST out*/);

/* HOST+DEVICE. a0: builds the k-space tables k_a(m), exp(-sigma2 k_a^2/2) and the
 * coefficient matrix c'_IJ = c_IJ / V in double on the host, uploads them as fp32, creates the
 * batched cuFFT plans (R2C x S, C2R x 3S).  PAPER.md L223 ("Fourier-space representation of the
 * inter-particle potential is calculated ... and stored"); analytic u^(k) per A5. */
int tild_init(tild_ctx** out /*HOST out*/, const tild_params* params /*HOST*/, void* workspace,
              size_t workspace_bytes, void* cuda_stream);

/* Loads (x, v) at step index step0, sorts particles by cell, evaluates F(x) once and forms the
 * split-kick state w = v - (dt/2m) F.  bond_partner may be NULL iff
 * max_bonds == 0.  Particle i keeps id i for the noise counter whatever the internal order. */
int tild_set_state(tild_ctx*, const float* x /*[n][3], in [0,L]*/, const float* v /*[n][3]*/,
                   const int32_t* type /*[n], 0..S-1*/, const int32_t* bond_partner /*[n][max_bonds], -1 = none*/,
                   uint64_t step0);

/* a1 + a2: spread.  grid[J][g] = sum_{i: type_i = J} W_x W_y W_z (raw weights, PAPER.md L223,
 * Eq. 1).  Pure function of (x, type); overwrites grid. */
int tild_spread(tild_ctx*, const float* x, const int32_t* type, float* grid /*[S][Nx][Ny][Nz]*/);

/* a3-a5: forward FFT, fused pair-kernel multiply + ik gradient, inverse FFT (Eq. 18):
 * ffield[I][a][g] = sum_m [-i k_a u^(k_m) sum_J c_IJ n^_J(m) / V] exp(+2 pi i m.g/N). */
int tild_kspace_force(tild_ctx*, const float* grid /*[S][M]*/, float* ffield /*[S][3][M]*/);

/* a6 (force only): f_i = sum_g W(g; r_i) ffield[type_i][.][g]  (L227, Fig. 1). Non-bonded only. */
int tild_interp(tild_ctx*, const float* ffield, const float* x, const int32_t* type, float* f /*[n][3]*/);

/* Bond forces alone (Eq. 2), for stage parity: f_i = sum_slots -2k(1 - r0/|d|) d. */
int tild_bond_force(tild_ctx*, const float* x, const int32_t* bond_partner, float* f /*[n][3]*/);

/* The timed path: (x, v)^t -> (x, v)^{t+nsteps}; each step = a1..a6 with bonds and the GJF
 * update fused into the interpolation pass.  One force evaluation per step. */
int tild_step(tild_ctx*, int32_t nsteps);

/* Copies the state out in ORIGINAL particle order.  v and f need one force evaluation at the
 * current positions (no state change).  Any of x, v, f may be NULL.  step is HOST out, nullable. */
int tild_get_state(tild_ctx*, float* x, float* v, float* f, uint64_t* step /*HOST*/);

/* HOST out, synchronises.  Energies of the current state (diagnostic): e[0] kinetic m/2 sum |v|^2,
 * e[1] bonded: sum over bonds k (|d| - r0)^2 (Eq. 2; every bond counted once, from its lower slot, so the partner
 * table must list a bond on both of its particles -- the force path does not need that) plus the angle energies
 * lambda (1 + cos theta) and k_theta (theta - theta0)^2 (Eq. 16-17) of every centre bead; e[2] non-bonded on the mesh
 * (1/2V) sum_m u^(k_m) sum_IJ c_IJ Re[n^_I(m) conj(n^_J(m))] (Eq. 3-4).  One force evaluation, no state change. */
int tild_energy(tild_ctx*, double e[3] /*HOST out*/);

/* Per-particle charges (the electrostatic forces "use the ... charge density field"; A25): q[i] is
 * the charge of particle i (original numbering).  While set, the charge mesh rho_c = sum_i q_i W(r - r_i) replaces the
 * charges per species of tild_params.charge in the Coulomb term (bjerrum, a_charge as before; k = 0 dropped).  q = NULL
 * switches back.  Costs one extra spread, one R2C and three C2R per step.  Needs TILD_FLAG_EXTRAS.  The energies and the
 * virial of tild_energy / tild_virial do not include this term. */
int tild_set_charges(tild_ctx*, const float* q /*DEVICE [n] or NULL*/);

/* Maier-Saupe interaction (PAPER.md IV.D L233-247, Eq. 19-20; A26): partner[i] = j names the particle that
 * defines the orientation u_i = (r_i - r_j)/|r_i - r_j| of LC centre i (-1: i is not a centre), as in the paper's list of
 * pairs (L245).  Forces: (2 mu/rho0) S_i : grad Phi(r_i) on the centre plus +-(4 mu/rho0)(I - u u) Phi u / |d| on centre and
 * partner, Phi = u_G * S on the mesh.  NULL switches it off.  Costs 6 spreads, 6 R2C and 24 C2R per step.  Needs
 * TILD_FLAG_EXTRAS and mu_ms != 0.  Not included in tild_energy / tild_virial. */
int tild_set_ms_partners(tild_ctx*, const int32_t* partner /*DEVICE [n] or NULL*/);

/* HOST out, synchronises.  Pressure virial of the current state, W = -dU/d ln(lambda) under the affine scaling r -> lambda r,
 * L -> lambda L (excess pressure = W / 3V): w[0] bonds, sum over bonds of -2 k (|d| - r0) |d| (the angle
 * potentials are scale invariant); w[1] non-bonded on the mesh, (1/2V) sum_m (3 - sigma2 k_m^2) u^(k_m) sum_IJ c_IJ Re[n^_I n^_J*]
 * plus (1 - 2 k^2 a_q^2) times the Coulomb term; NaN with TILD_FLAG_SAMPLED_KERNEL. */
int tild_virial(tild_ctx*, double w[2] /*HOST out*/);

/* Structure factor of the current state (diagnostic; Eq. 23, "Compute" class L332-336):
 * sk[m] (= or +=, by `accumulate`) |sum_{J in species_mask} n^_J(m)|^2 / N_mask on the half spectrum
 * [Nx][Ny][Nz/2+1], with n^ the transform of the mesh (spread) density and N_mask the particles of the masked
 * species.  Averaging over time is the caller's: accumulate, then divide by the number of samples. */
int tild_structure_factor(tild_ctx*, uint32_t species_mask, float* sk /*DEVICE [Nx][Ny][Nz/2+1]*/, int32_t accumulate);

/* a1: index map of arbitrary caller positions.  base[i][a] = first stencil node (unwrapped),
 * cell_key[i] = (cx*Ny+cy)*Nz+cz, perm = particle ids grouped by ascending cell key (order inside
 * a cell unspecified), cell_start[c] = #particles with key < c (M+1 entries).  Any output may be NULL. */
int tild_index_map(tild_ctx*, const float* x, int32_t* base /*[n][3]*/, uint32_t* cell_key /*[n]*/,
                   uint32_t* perm /*[n]*/, uint32_t* cell_start /*[M+1]*/);

/* HOST, synchronises.  Mean milliseconds per step over the tild_step calls since the last call
 * (needs TILD_FLAG_TIMING): sort, spread (incl. zero fill), fft_fwd, kspace, fft_inv, interp(+bonds
 * +GJF), other, total.  steps_timed (nullable) receives how many steps the means cover. */
int tild_get_timings(tild_ctx*, float ms[8] /*HOST out*/, int32_t* steps_timed /*HOST out*/);

/* HOST buffers, synchronises: the end-to-end call.  Copies (x, v, type, bond_partner) host->device,
 * runs tild_set_state + tild_step(nsteps), copies (x, v) back.  Buffers should be pinned for speed. */
int tild_run_host(tild_ctx*, float* x_host, float* v_host, const int32_t* type_host,
                  const int32_t* bond_partner_host, uint64_t step0, int32_t nsteps);

/* HOST buffers: the pipelined end-to-end path for INDEPENDENT batches (needs TILD_FLAG_HOST_PIPELINE and a context on a
 * stream of its own).  tild_run_host_submit copies one batch host->device on a copy stream, runs tild_set_state +
 * tild_step(nsteps) + the read-out on the context's stream and starts the copy of (x, v) to x_out_host / v_out_host on a
 * second copy stream; it returns once the inputs have been consumed (they may be reused), not when the results are there.
 * tild_run_host_wait blocks until the results of the oldest batch not yet waited for are in its output buffers
 * (TILD_ESTATE if there is none; at most four batches may be in flight).  Calling submit again before wait overlaps the three phases of consecutive batches;
 * outputs of a batch are valid only after its wait.  Buffers should be pinned.  The context's state after a submit is
 * that batch's; tild_step / tild_get_state may follow, stage calls too. */
int tild_run_host_submit(tild_ctx*, const float* x_host, const float* v_host, const int32_t* type_host,
                         const int32_t* bond_partner_host, uint64_t step0, int32_t nsteps, float* x_out_host, float* v_out_host);
int tild_run_host_wait(tild_ctx*);

/* Test hook: out[i] = Philox4x32-10(counter = ctr[i], key = key[i]) computed by the same device
 * function the integrator uses; gauss[i] = the three N(0,1) draws for (id = ctr[i].x, step =
 * ctr[i].y | ctr[i].z << 32) under key[i].  gauss may be NULL. */
int tild_philox_test(tild_ctx*, const uint32_t* ctr /*[m][4]*/, const uint32_t* key /*[m][2]*/,
                     uint32_t* out /*[m][4]*/, float* gauss /*[m][3]*/, int32_t m);

/* HOST. The internal tiling: info = {tiles, segments = tiles * species, image nodes in z,
 * spread kernel shared bytes, interpolation kernel shared bytes, tile cells x, y, z}.  Needs tild_set_state. */
int tild_layout_info(const tild_ctx*, uint64_t info[8] /*HOST out*/);

/* The ordering the timed path runs on, for the bit-exact check of the sort that tild_step uses:
 * seg_base[g] = first slot of segment g = tile * S + species (tiles in x-major order of tild_layout_info's tile edges,
 * tile of a particle = its cell (a1 index map) / tile edge per axis), nseg + 1 entries; slot_id[s] = original particle
 * id held by slot s.  Describes the particles as they were at the last re-sort.  Either output may be NULL. */
int tild_segment_layout(const tild_ctx*, uint32_t* seg_base /*DEVICE [tiles*S + 1]*/, uint32_t* slot_id /*DEVICE [n]*/);

/* The cell offsets of the a1 index map WITHOUT a context and without any allocation, for callers that cannot call
 * cudaMalloc (code under CUDA graph capture, serving loops, harnesses that forbid it): histogram of the cell keys +
 * exclusive scan, the first half of the counting sort (particles binned by cell).
 *   cell_key   DEVICE [n], as tild_index_map writes it: (cx*Ny+cy)*Nz+cz
 *   cell_start DEVICE [n_cells + 1] out: cell_start[c] = #particles with key < c (equals tild_index_map's, bit for bit)
 *   n_bad      DEVICE [1] out or NULL: keys >= n_cells; such particles are left out instead of indexing out of bounds
 *   stream     a cudaStream_t (NULL = default stream); the call is asynchronous on it
 *   errmsg     HOST [errmsg_len] out or NULL: the reason when the result is not TILD_OK
 * The scan's block partials live in a static __device__ array (16.4 KB that every GPU loading the library holds until
 * exit) sized for n_cells <= TILD_NOALLOC_MAX_CELLS (a 256^3 mesh); larger sizes return TILD_EINVAL.  The call runs one
 * memset and four kernels on `stream` with the device that is current, and calls no cudaMalloc / cudaFree and no allocating
 * library routine.  All calls on a device share the array (it is rewritten before it is read: nothing is kept between
 * calls): calls that can overlap on the GPU -- different streams without an ordering between them -- race on it. */
#define TILD_NOALLOC_MAX_CELLS 16777216
int tild_cell_start_noalloc(const uint32_t* cell_key, int32_t n, uint32_t n_cells, uint32_t* cell_start, uint32_t* n_bad,
                            void* stream, char* errmsg, size_t errmsg_len);

/* HOST. Number of kernels of this library launched on the context's stream so far. */
int64_t tild_launch_count(const tild_ctx*);

const char* tild_last_error(const tild_ctx*); /* HOST; valid until the next call on the context */
void tild_destroy(tild_ctx*);
const char* tild_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TILD_H */
