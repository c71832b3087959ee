/*
 * gf.h — C ABI of libgf.so: SU(3) (and SU(2)) lattice gauge fixing by checkerboard local updates on one B200.
 *
 * The operations are those of Schroeck & Vogt, "Coulomb, Landau and Maximally Abelian Gauge Fixing
 * in Lattice QCD with Multi-GPUs" (arxiv 1212.5221; line numbers below refer to the text of the
 * paper as PAPER.md).  Every entry point enqueues hand-written sm_100a CUDA kernels; there is no
 * CPU fallback: without a CUDA device gf_create fails with GF_ECUDA.
 *
 * Conventions common to all calls
 *   - Return value: 0 = GF_OK, 1 = GF_NOT_CONVERGED (gf_run, gf_run_batch, gf_fix), < 0 = error.  No exception or
 *     abort crosses the ABI.  gf_last_error(ctx) returns a ctx-owned, NUL-terminated description of
 *     the last error (valid until the next call on that ctx).
 *   - A context owns all of its device memory.  The caller owns every pointer it passes in; the
 *     library never keeps a caller pointer beyond the call.
 *   - A context holds one lattice (gf_create) or n_copies lattices of the same extents (gf_create_batch), of
 *     the gauge group SU(3) or, with GF_FLAG_SU2, SU(2).
 *   - A context lives on the CUDA device that is current when it is created; the caller keeps that device
 *     current for every later call on the context.
 *   - One context per stream.  A context is not thread-safe, but different contexts may be driven from different
 *     host threads at the same time (the library keeps no unguarded global state).  Kernels are enqueued on the cudaStream_t given to
 *     gf_create (NULL = the legacy default stream).  gf_set_links, gf_get_*, gf_measure*, gf_run*, gf_fix,
 *     gf_random_gauge, gf_plaquette and gf_unitarity synchronise that stream before returning; gf_sweep,
 *     gf_half_sweep, gf_anneal, gf_wilson_heatbath, gf_reunitarize and gf_coulomb_finalize only enqueue.
 *   - Host-side link layout ("StandardPattern", Sec. 4.2.1; mu = 0 is the temporal
 *     direction): links[t][x][y][z][mu][i][j][c], c = 0 real / 1 imaginary, i.e. real
 *     offset ((((((t*Nx + x)*Ny + y)*Nz + z)*4 + mu)*3 + i)*3 + j)*2 + c.  mu = 1,2,3 are x,y,z.
 *     Gauge transforms use [t][x][y][z][i][j][c].
 *   - All four extents must be even and >= 2 (the red/black colouring of PAPER.md:293 fn. 3 is
 *     inconsistent under periodic boundaries otherwise); Nx*Ny*Nz*Nt < 2^32.
 */
#ifndef GF_H_
#define GF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gf_ctx gf_ctx; /* opaque */

/* return codes */
#define GF_OK 0
#define GF_NOT_CONVERGED 1 /* gf_run / gf_run_batch / gf_fix: max_sweeps reached before every unit had theta < eps */
#define GF_EINVAL (-1) /* bad argument (odd extent, unknown gauge/algo, NULL pointer, ...) */
#define GF_ENOMEM (-2) /* device or host allocation failed */
#define GF_ECUDA (-3)  /* a CUDA runtime call or kernel launch failed; see gf_last_error */
#define GF_ESTATE (-4) /* call not valid in this state (e.g. no links set, transform not tracked) */

/* precision policy (Sec. 4.5) */
#define GF_SP 0 /* float links, float Step 1 and Step 2; reductions and reunitarisation in double */
#define GF_DP 1 /* everything in double */
#define GF_MP 2 /* float links and Step 2; Step 1 (gauge-update calculation) in double */

/* gauge (Sec. 2.1) */
#define GF_LANDAU 0  /* Eq. (4), all four directions */
#define GF_COULOMB 1 /* Eq. (4) restricted to mu = 1,2,3; every time-slice is its own problem */
#define GF_MAG 2     /* maximally Abelian gauge, functional Eq. (11) */

/* Step-1 update rule (Secs. 2.2.3-2.3) */
#define GF_OR 0    /* overrelaxation g -> g^omega "to first order" = Fig. A.11; param = omega in [1,2) */
#define GF_SR 1    /* stochastic relaxation: g^2 with probability param = p, else g */
#define GF_SA 2    /* simulated-annealing heatbath at temperature param = T; its arithmetic is double on
                      GF_DP / GF_MP contexts and float on GF_SP contexts, where every accept/reject decision that float
                      cannot settle is re-evaluated in double */
#define GF_MICRO 3 /* microcanonical step g -> g^2; param ignored */

/* gf_create flags */
#define GF_FLAG_TRACK_TRANSFORM 1u /* accumulate g(x) so that gf_get_gauge_transform / Coulomb finalisation work */
#define GF_FLAG_SU2 4u /* gauge group SU(2) instead of SU(3) (Eqs. (8), (12)-(15), (20)-(29)); see "SU(2)" below */
#define GF_FLAG_FREEZE_SLICES 2u   /* gf_run(Coulomb): stop sweeping a time-slice once its own theta_t < eps */
#define GF_FLAG_LAGGED_STOP 8u     /* gf_run: take the stopping decision half a sweep late at no cost; see gf_run */

/*
 * gf_create — allocate a context for an Nx*Ny*Nz*Nt periodic lattice (BASELINE.json north_star:
 * gf_create(Nx,Ny,Nz,Nt,precision)).  recon = 18 stores full links, recon = 12 stores the first two
 * rows and rebuilds the third as (u x v)^* on load.  Device storage is parity-split
 * structure-of-arrays in 16-byte vectors.  cuda_stream: a cudaStream_t or NULL.
 * Errors: GF_EINVAL (extents, precision, recon), GF_ECUDA (no device), GF_ENOMEM.
 */
int gf_create(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int precision, int recon, unsigned flags,
              void* cuda_stream);
int gf_destroy(gf_ctx* ctx);

/*
 * SU(2) (contexts created with GF_FLAG_SU2).  The paper states its local problems
 * for SU(2) — Eq. (20) for Landau/Coulomb, Eqs. (21)-(29) for the maximally
 * Abelian gauge, theta of Eqs. (12)-(13) — and reaches SU(3) through the SU(2) subgroups;
 * with this flag the links themselves are SU(2) matrices and Step 1 acts once, on the whole group.  Every
 * call keeps its meaning with N_c = 2 in Eqs. (4), (7), (11), (13).  Host layouts become
 * links[t][x][y][z][mu][i][j][c] and g[t][x][y][z][i][j][c] with i,j in {0,1} (8 reals per matrix); only
 * the first row (u0 + i u3, u2 + i u1) of Eq. (15) is read, the device keeps those four reals
 * per link (one float4 / two double2; `recon` is ignored) and the second row returned is (-conj b, conj a).
 * gf_num_colors returns N_c (3 or 2).
 */
int gf_num_colors(const gf_ctx* ctx);

/*
 * Batched gauge copies.  The paper's production use fixes many gauge copies
 * of one configuration — "100 randomly chosen points on the gauge orbit" — and
 * a 32^4 or smaller lattice does not fill a B200.  gf_create_batch makes a context that holds
 * n_copies independent lattices of the same extents (contiguous in HBM, each in the layout of
 * gf_create); every sweep / reduction / reunitarisation launch then covers all copies
 * (grid.y = n_copies * Nt, so n_copies * Nt <= 65535).  Copy c draws its random numbers with the
 * Philox key seed + c, so its trajectory is that of a single-lattice context run with seed + c.
 * gf_create(...) == gf_create_batch(..., n_copies = 1, ...).
 *
 * On a batch context gf_set_links stores the same configuration into every copy; gf_sweep,
 * gf_half_sweep, gf_anneal, gf_reunitarize, gf_coulomb_finalize and gf_random_gauge act on all copies;
 * gf_get_links, gf_get_gauge_transform, gf_measure and gf_run need n_copies == 1 (else GF_ESTATE) —
 * use the _copy / _batch forms below, which are valid for any n_copies.
 */
int gf_create_batch(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int n_copies, int precision, int recon,
                    unsigned flags, void* cuda_stream);
int gf_num_copies(const gf_ctx* ctx);
int gf_set_links_copy(gf_ctx* ctx, int copy, const void* links, int elem_bytes, int is_device);
int gf_get_links_copy(gf_ctx* ctx, int copy, void* links, int elem_bytes, int is_device);
int gf_get_gauge_transform_copy(gf_ctx* ctx, int copy, void* g, int elem_bytes, int is_device);

/*
 * gf_set_links / gf_get_links — copy a whole configuration in / out in StandardPattern.
 * links: host pointer (is_device = 0) or device pointer (is_device = 1) to Nt*Nx*Ny*Nz*4*18 reals of
 * elem_bytes = 4 (float) or 8 (double), independent of the context's precision (converted on the
 * way).  gf_set_links resets the accumulated gauge transform to the identity.  With recon = 12 the
 * third row returned by gf_get_links is the reconstructed one.  Synchronous.
 */
int gf_set_links(gf_ctx* ctx, const void* links, int elem_bytes, int is_device);
int gf_get_links(gf_ctx* ctx, void* links, int elem_bytes, int is_device);

/*
 * gf_get_gauge_transform — the accumulated g(x) with U_now = g(x) U_set g(x+mu)^dagger (Eq. (1),
 * PAPER.md:25), layout [t][x][y][z][i][j][c].  Needs GF_FLAG_TRACK_TRANSFORM (else GF_ESTATE).
 */
int gf_get_gauge_transform(gf_ctx* ctx, void* g, int elem_bytes, int is_device);

/*
 * gf_sweep — one sweep of Alg. 1: the even half-sweep then the odd one.  For every
 * site x of the active parity: gather U_mu(x), U_mu(x-mu); for the SU(2) subgroups (0,1),(0,2),(1,2)
 * find g (Step 1, rule `algo`) and rotate U_mu(x) <- g U_mu(x), U_mu(x-mu) <- U_mu(x-mu) g^dagger
 * (Step 2).  Parity is (t+x+y+z)&1 for Landau/MAG and (x+y+z)&1 in every time-slice
 * for Coulomb, whose sweeps touch spatial links only.
 * seed / sweep_index key the counter-based Philox4x32-10 generator (PAPER.md:249 fn. 2) as
 * counter = (lexicographic site index, sweep_index, subgroup | purpose << 8, trial), key = seed;
 * they are ignored by GF_OR and GF_MICRO.  Asynchronous.
 * gf_half_sweep does one parity only (parity 0 = even, 1 = odd).
 */
int gf_sweep(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t sweep_index);
int gf_half_sweep(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t sweep_index,
                  int parity);

/*
 * gf_measure — gauge functional F (Eq. (4), N_d = 3 for Coulomb; Eq. (11) PAPER.md:102 for
 * MAG) and gauge precision theta (Eq. (7); MAG: sum over the three subgroups of
 * |X^s_12|^2 / (N_c V), R11), reduced on the device in double with a fixed summation order
 * (bit-reproducible).  theta_slice: NULL or Nt doubles receiving theta of every time-slice
 * (V -> Nx*Ny*Nz), the Coulomb stopping quantity.  Synchronous.
 */
int gf_measure(gf_ctx* ctx, int gauge, double* F, double* theta, double* theta_slice);
/* the same for every copy: F[n_copies], theta[n_copies], theta_slice NULL or [n_copies][Nt] */
int gf_measure_batch(gf_ctx* ctx, int gauge, double* F, double* theta, double* theta_slice);
/*
 * gf_measure_mag_eq16 — the maximally Abelian precision as Eq. (16) prints it for SU(3),
 * theta_eq16[c] = 1/(N_c V) sum_x |X_12 + Y_12 + Z_12|^2 for every copy c, the sum over the three SU(2) subgroups INSIDE
 * the modulus.  gf_measure / gf_run use sum_x sum_s |X^s_12|^2 / (N_c V) instead (R11): a norm, zero exactly
 * at a stationary point, whereas the printed form can vanish away from one; theta_eq16 <= 3 theta, and the two differ by
 * the cross terms.  eps thresholds and MAG theta values quoted from the paper (Table 4, Fig. 7) refer to the printed
 * form: compare them with this call.  SU(3) contexts only (GF_ESTATE otherwise).  Synchronous.
 */
int gf_measure_mag_eq16(gf_ctx* ctx, double* theta_eq16);

typedef struct {
    int sweeps;   /* sweeps performed */
    double F;     /* functional at the last check */
    double theta; /* stopping quantity at the last check: theta, or max_t theta_t for Coulomb */
} gf_result;

/*
 * gf_run — Alg. 1's outer loop: sweep (sweep s uses sweep_index first_sweep_index + s)
 * until the stopping quantity < eps, checked after every check_every-th sweep and after the last one,
 * or until max_sweeps.  reunit_every > 0 reprojects all links (and the tracked transform) onto SU(3)
 * after every reunit_every-th sweep.  hist: NULL or room for
 * 3 * (max_sweeps / check_every + 1) doubles, filled with (sweep, F, theta) per check.
 * For Coulomb with a tracked transform the temporal links are finalised before returning
 * (PAPER.md:448).  Returns GF_OK if converged, GF_NOT_CONVERGED otherwise.  Synchronous.
 *
 * Cost of a check: the odd half-sweep of a check sweep s leaves F(s) and the odd sites' share of theta(s), a lower
 * bound of theta(s), at no extra traffic; only a check at which that bound is below eps runs the stand-alone
 * reduction (one read of every link twice, about one half-sweep), so every stopping decision is the one a reduction
 * after every check would take (Alg. 1).  With GF_FLAG_LAGGED_STOP (single lattice, GF_DP or GF_MP, not
 * with GF_FLAG_FREEZE_SLICES; ignored on GF_SP contexts, whose fused sums are formed in float and carry ~1e-12 of
 * rounding noise in theta: they keep the stand-alone reduction) that reduction is not run either: the even sites' share of theta(s) is what the even
 * half-sweep of sweep s + 1 sees before it updates, so theta(s) is known, exactly and at no cost, half a sweep later.
 * If theta(s) < eps the run stops THERE: out->sweeps = s, and the links returned have received the even half-sweep of
 * sweep s + 1 on top of Alg. 1's s sweeps (out->F, out->theta are those of the links returned; GF_OK).  A check at
 * max_sweeps is decided by the stand-alone reduction as without the flag.  The oracle's run loop mirrors this reading
 * (oracle/gf_oracle.py, lagged_stop).
 */
int gf_run(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t first_sweep_index,
           int max_sweeps, double eps, int check_every, int reunit_every, gf_result* out, double* hist);
/*
 * gf_run_batch — gf_run for every copy of a batch context in the same launches.  Every copy is its own
 * optimisation problem: copy c is no longer swept after the first check at which its stopping quantity
 * is < eps (its CTAs exit at once), so out[c] (n_copies entries) is what gf_run returns for a
 * single-lattice context holding copy c (seed + c).  hist: NULL or 3 * n_copies * (max_sweeps /
 * check_every + 1) doubles, entry (check k, copy c) at hist[3 * (k * n_copies + c)]; a stopped copy
 * repeats its final values.  GF_OK if every copy converged, else GF_NOT_CONVERGED.
 */
int gf_run_batch(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t first_sweep_index,
                 int max_sweeps, double eps, int check_every, int reunit_every, gf_result* out, double* hist);

/*
 * Per-slice Coulomb fixing (contexts created with GF_FLAG_FREEZE_SLICES).  In Coulomb gauge every
 * time-slice is an independent optimisation problem and the paper fixes them one at a
 * time.  Here all slices are swept in the same launches, and gf_run(GF_COULOMB) stops
 * sweeping slice t at the first check at which theta_t < eps (the CTAs of a stopped slice exit at
 * once), so the result of slice t is that of a stand-alone run on that slice.  gf_run then returns
 * GF_OK when every slice has stopped; out->theta = max_t theta_t of the final links.  Reprojection
 * (reunit_every) still covers all links, stopped slices included: on float-storage contexts (GF_SP, GF_MP) a slice
 * that stopped with theta_t < eps is rounded to float again by every later reprojection and may then read up to
 * about 3 eps at the final measurement for eps near the float floor (1e-10); the stopping decision itself was taken
 * on theta_t < eps, and GF_DP contexts return theta_t < eps for every slice.  Landau/MAG runs ignore the flag.
 * gf_get_slice_sweeps: sweeps[n_copies * Nt] (host) receives the number of sweeps applied to every slice
 * of every copy by the last gf_run / gf_run_batch (without the flag or for other gauges: the sweep count
 * of the slice's copy in every entry).
 * GF_ESTATE before the first gf_run.
 */
int gf_get_slice_sweeps(gf_ctx* ctx, int* sweeps);

/*
 * gf_anneal — simulated annealing schedule: n_steps heatbath sweeps at
 * T_k = T_hi - k (T_hi - T_lo)/(n_steps - 1), each followed by n_micro microcanonical sweeps; every
 * sweep consumes one sweep index starting at first_sweep_index.  *next_sweep_index (may be NULL)
 * receives the first unused index.  Asynchronous.
 * On contexts with recon = 12 the links are reprojected onto SU(3) after every 16th sweep of the schedule (the
 * rebuilt third row compounds the norm errors of the two stored rows under large rotations: |1 - det U| grows by
 * about a third per heatbath or microcanonical sweep).  gf_fix does the same in its annealing and
 * stochastic-relaxation stages, and gf_run / gf_run_batch with GF_SA, GF_MICRO or GF_SR on such a context use
 * reunit_every = 16 when asked for none or for a longer interval.  (Sequences of single gf_sweep calls are the
 * caller's: call gf_reunitarize.)
 */
int gf_anneal(gf_ctx* ctx, int gauge, double T_hi, double T_lo, int n_steps, int n_micro, uint64_t seed,
              uint32_t first_sweep_index, uint32_t* next_sweep_index);

/*
 * gf_fix — the paper's production recipe as one call: (1) sa_steps steps of
 * simulated annealing from sa_T_hi down to sa_T_lo (gf_anneal's schedule, sa_micro microcanonical sweeps
 * after every heatbath sweep), (2) at most sr_max_sweeps sweeps of stochastic relaxation with probability
 * sr_p, (3) overrelaxation with or_omega until theta < eps or or_max_sweeps.  A stage of length 0 is left
 * out.  Stages (2) and (3) are gf_run_batch loops (checks every check_every sweeps; a copy that reaches
 * theta < eps is stopped and takes no part in later stages); reunit_every > 0 reprojects after every
 * reunit_every-th sweep of each stage.  Sweep indices run on from stage to stage starting at 0; copy c
 * uses the Philox key seed + c.  out[n_copies]: total sweeps of all stages, F and the stopping quantity
 * of the final links.  GF_OK if every copy converged, else GF_NOT_CONVERGED.  Synchronous.
 */
typedef struct {
    int gauge;
    uint64_t seed;
    int sa_steps;
    double sa_T_hi, sa_T_lo;
    int sa_micro;
    int sr_max_sweeps;
    double sr_p;
    double or_omega;
    int or_max_sweeps;
    double eps;
    int check_every, reunit_every;
} gf_fix_params;
int gf_fix(gf_ctx* ctx, const gf_fix_params* params, gf_result* out);

/*
 * t-shards: one lattice split along t over several link stores (Sec. 5).
 *
 * The paper splits N_t over the devices; the only links a half-sweep touches outside its own part
 * are the inactive-parity U_0 of the boundary slice, 1/12 of a slice.  gf_create_shard makes a
 * context that holds the slices [t0, t0 + Nt_local) of an Nx*Ny*Nz*Nt_global lattice (t0 and both extents even; SU(3),
 * one gauge copy).  Its half-sweep kernel reads and writes the down-t links of its first slice IN PLACE in the store
 * of the shard below — a pointer on the same device, a peer mapping (gf_shard_attach: contexts of this process, peer
 * access is enabled when they live on another device) or a CUDA IPC mapping (gf_shard_export / gf_shard_attach_ipc:
 * other processes) — so there are no halo buffers and no exchange step (the seven steps of PAPER.md:454-463 collapse
 * into the kernel's own loads and stores over NVLink).  Every link is still touched by exactly one thread per
 * half-sweep.  The Philox counter uses the site index in the WHOLE lattice and the reductions are summed per global
 * time-slice in slice order on every shard, so links, F, theta, histories, stopping decisions and random draws are
 * those of the unsharded context, bit for bit.
 *
 * What is left between shards is ordering and 2*Nt_global numbers per check (gf_comm, supplied by the caller — the
 * library links no communication library):
 *   barrier(user)              stream-ordered barrier over all shards: whatever was enqueued before it on any shard's
 *                              stream completes before anything enqueued after it on any shard's stream starts.  Called
 *                              after every Landau/MAG half-sweep and reprojection, before a reduction, around the
 *                              Coulomb finalisation and after gf_set_links; Coulomb sweeps need none.
 *                              One stream shared by all shards of a device: a no-op.  One process per GPU: an
 *                              all-reduce of one element enqueued on the context's stream (NCCL).
 *   allreduce_sum(user, b, n)  in-place sum over all shards of the host array b[n] (every shard has filled its own
 *                              slices and zeroed the rest, so the sum is exact); blocking.
 * Every shard must make the same sequence of calls with the same arguments (they take identical decisions).
 * On a shard: gf_set_links / gf_get_links / gf_get_gauge_transform move the shard's own slab
 * [t0, t0 + Nt_local) (contiguous in StandardPattern: t is the slowest index); gf_measure returns the global F and
 * theta, theta_slice has Nt_global entries; gf_run / gf_anneal / gf_fix / gf_sweep / gf_half_sweep / gf_reunitarize /
 * gf_coulomb_finalize (which reads g(x + t_hat) of its last slice from the shard above) work as on a
 * whole lattice, and so does gf_random_gauge (h(x) is a function of the site index in the whole lattice: a shard
 * recomputes h of the slice above for its last temporal links); gf_get_slice_sweeps has Nt_global entries;
 * gf_unitarity covers the shard's own links; gf_plaquette returns the plaquette of the whole lattice (the last slice
 * reads the first one of the store above); gf_wilson_heatbath returns GF_ESTATE.  Sweeps and reductions return GF_ESTATE
 * until the neighbours are attached.  A single shard spanning the lattice attaches to itself.
 * The tests drive 2 and 4 shards on one device — threads of one process, and two processes with IPC-mapped stores —
 * and compare with the unsharded context bit for bit; mappings of ANOTHER device's memory were not run in this build
 * (one GPU available).
 */
int gf_create_shard(gf_ctx** out, int Nx, int Ny, int Nz, int Nt_local, int t0, int Nt_global, int precision, int recon,
                    unsigned flags, void* cuda_stream);
/* below holds slice t0 - 1 as its last slice, above holds slice t0 + Nt_local as its first one (periodic in Nt_global) */
int gf_shard_attach(gf_ctx* ctx, gf_ctx* below, gf_ctx* above);
typedef struct {
    unsigned char links[64], gtot[64], gapplied[64]; /* cudaIpcMemHandle_t of the stores */
    int t0, Nt_local, has_transform;
    int Nx, Ny, Nz, Nt_global, precision, recon;     /* what the store was created with: checked by gf_shard_attach_ipc */
} gf_shard_handle;
int gf_shard_export(gf_ctx* ctx, gf_shard_handle* handle);
int gf_shard_attach_ipc(gf_ctx* ctx, const gf_shard_handle* below, const gf_shard_handle* above);
typedef struct {
    void (*barrier)(void* user);
    void (*allreduce_sum)(void* user, double* buf, int n);
    void* user;
} gf_comm;
/*
 * gf_shard_attach_ipc maps the neighbours' stores only after checking that they were created with this shard's extents,
 * precision, recon and Nt_global, that they adjoin its slices and that all three track a transform or none does
 * (GF_EINVAL otherwise, nothing mapped).  A call that fails part-way closes what it had opened, and a repeated call
 * closes the previous mappings first.  gf_shard_attach (same process) refuses neighbours that live on this shard's
 * device but use another stream, unless a communicator with a barrier has been set BEFORE the attach: a barrier that
 * only synchronises host threads orders nothing between two streams.
 */
/* comm == NULL: no communicator (all shards on one stream of one process need none for ordering, but still need
 * allreduce_sum for reductions unless there is a single shard) */
int gf_shard_set_comm(gf_ctx* ctx, const gf_comm* comm);
int gf_shard_info(const gf_ctx* ctx, int* t0, int* Nt_local, int* Nt_global);

/*
 * gf_random_gauge — a random start on the gauge orbit ("100 randomly chosen points on the
 * gauge orbit", 580): every copy c is gauge transformed, U_mu(x) <- h(x) U_mu(x) h(x+mu)^dagger (Eq. (1),
 * PAPER.md:25), with h(x) Haar distributed on SU(3): two rows of complex standard normals — Box-Muller on
 * the Philox uniforms of counter (site, 0, k | 3 << 8, 0), k = 0,1,2, key seed + c: normals 4k..4k+3 =
 * sqrt(-2 ln u0) (cos, sin)(2 pi u1), sqrt(-2 ln u2) (cos, sin)(2 pi u3) — orthonormalised by
 * Gram-Schmidt, third row (u x v)^* (R27), all in double.  A tracked transform is updated,
 * g(x) <- h(x) g(x).  Synchronous.
 */
int gf_random_gauge(gf_ctx* ctx, uint64_t seed);

/*
 * Input generator.  The paper's production input is a thermalised beta = 5.7 32^4
 * configuration of the Wilson gauge action, which is not distributed with it.
 * gf_wilson_heatbath runs n_sweeps Cabibbo-Marinari pseudo-heatbath sweeps (the SU(2)-subgroup method of the
 * paper's ref. [31]) of S = beta sum_P (1 - Re tr U_P / N_c) on every copy of a context (SU(3) in what follows): for mu = 0..3,
 * for parity even, odd, every link U_mu(x) of that parity is multiplied from the left, subgroup by subgroup
 * ((0,1),(0,2),(1,2)), by g drawn with P(g) ~ exp((beta/3) Re tr[g~ U A]), A the sum of the six staples
 * (Kennedy-Pendleton / Creutz sampler of GF_SA at T = 3/beta).  Philox counter (site, 4 * sweep + mu,
 * sub | purpose << 8, trial), key seed + copy, sweeps first_sweep_index .. first_sweep_index + n_sweeps - 1.
 * The result is a new configuration, so a tracked transform restarts at the identity.  Asynchronous.
 * On contexts with recon = 12 the links are reprojected onto SU(3) after every 16th sweep of the call (as in gf_anneal),
 * on other float contexts after every 100th.  On contexts with float storage (GF_SP and GF_MP) the
 * heatbath arithmetic of this generator is float with guard-banded accept decisions (the kernel works in
 * the storage type, so GF_MP does not buy a double heatbath here as it does in GF_SA sweeps).
 * On SU(2) contexts the same with the single subgroup and the weight exp((beta/2) Re tr[U A]) (T = 2/beta).
 * gf_plaquette: plaq[n_copies] receives <Re tr U_P> / N_c over the 6 V plaquettes (gauge invariant under
 * Eq. (1): it does not change under any sweep of this library).  Synchronous.
 */
int gf_wilson_heatbath(gf_ctx* ctx, double beta, uint64_t seed, uint32_t first_sweep_index, int n_sweeps);
int gf_plaquette(gf_ctx* ctx, double* plaq);

/*
 * gf_unitarity — the unitarity measure of Eq. (33): avg[c] = (1/4V) sum_{mu,x} |1 - det U_mu(x)| and
 * max[c] = max_{mu,x} |1 - det U_mu(x)| for every copy c (n_copies entries each, either may be NULL), evaluated in
 * double from the stored links (recon = 12: with the rebuilt third row; SU(2): det U = |u|^2 of the stored quaternion).
 * Synchronous.
 */
int gf_unitarity(gf_ctx* ctx, double* avg, double* max);

/*
 * gf_unitarity_noalloc — the same measure, Eq. (33), for callers that must not allocate: no context,
 * and no cudaMalloc, cudaFree or other allocating call inside, on any call.
 *
 * Why it exists: gf_unitarity needs a context, i.e. a second copy of the configuration on the GPU, and it takes and
 * frees two scratch buffers per call (the cudaFree waits for the whole device).  A lattice code whose own fields
 * already fill the GPU, code that lives inside a memory pool with a fixed budget, or a monitoring step that must not
 * stall the kernels of other streams cannot use that; here they hand in the buffer they already have.
 *
 *   links_device   DEVICE pointer to n_links SU(3) matrices of 18 reals each, row major with re/im innermost (one
 *                  link of the StandardPattern host layout above; a whole configuration in that layout is
 *                  n_links = 4 V).  Read only; aligned to 2 * elem_bytes.  The link order plays no role.
 *   elem_bytes     4 (float) or 8 (double); the determinant is evaluated in double either way.
 *   n_links        0 <= n_links <= GF_UNITARITY_NOALLOC_MAX_LINKS (2^28 = the 4 V links of 64^3 x 256).  More is
 *                  rejected with GF_EINVAL: measure the buffer in pieces and combine the averages and maxima.
 *   result_device  DEVICE pointer to 2 doubles owned by the caller: [0] = (1/n_links) sum |1 - det U|, [1] = max
 *                  |1 - det U| (both 0 for n_links = 0).  Valid once the work enqueued on cuda_stream has finished.
 *   cuda_stream    a cudaStream_t or NULL.  The call only enqueues two kernels there (asynchronous).
 *   errbuf         NULL, or errbuf_len bytes that receive a NUL-terminated description when the return value is not
 *                  GF_OK (there is no context whose gf_last_error could hold it).
 * Errors: GF_EINVAL (arguments, size, alignment — checked before the device is touched), GF_ECUDA.
 *
 * The scratch memory — one (sum, max) pair per 2048 links — is a fixed array inside libgf.so's device image, 2 MiB
 * on every GPU that loads the library, held until the process exits.  Consequences:
 *   - All calls on one device share it.  Calls whose kernels may overlap on the GPU (different streams or host
 *     threads without an ordering between them) corrupt each other's result; calls on one stream are safe, and so
 *     are calls on different devices.  Nothing has to be zeroed between calls: every entry a call reads it has
 *     written itself, whatever the previous call left behind.
 *   - The first call on each device (with that device current, as for every call) looks up the array's address on
 *     that device; make that first call before you start capturing a stream.
 */
#define GF_UNITARITY_NOALLOC_MAX_LINKS (1 << 28)
int gf_unitarity_noalloc(const void* links_device, int elem_bytes, int64_t n_links, double* result_device,
                         void* cuda_stream, char* errbuf, int errbuf_len);

/*
 * gf_reunitarize — reproject every link (and the tracked transform) onto SU(3): Gram-Schmidt on rows
 * 0,1 in double, third row (u x v)^* (R20).  Asynchronous.
 */
int gf_reunitarize(gf_ctx* ctx);

/*
 * gf_coulomb_finalize — apply the accumulated g to the temporal links,
 * U_0(x,t) <- g(x,t) U_0(x,t) g(x,t+1)^dagger.  Idempotent: only the part of g not yet
 * applied is used.  Called implicitly by gf_run(Coulomb), gf_get_links and by Landau/MAG calls that
 * follow Coulomb sweeps.  Needs GF_FLAG_TRACK_TRANSFORM (else GF_ESTATE).  Asynchronous.
 */
int gf_coulomb_finalize(gf_ctx* ctx);

/* gf_sync — wait for everything enqueued on the context's stream. */
int gf_sync(gf_ctx* ctx);

/*
 * gf_kernel_time_ms — device time (CUDA events on the context's stream) of the half-sweep kernels
 * launched since the last call with reset != 0: *total_ms receives their summed duration, *launches
 * their count.  Timing is off until gf_kernel_timing(ctx, 1).  Used by bench.py for the roofline.
 */
int gf_kernel_timing(gf_ctx* ctx, int enable);
int gf_kernel_time_ms(gf_ctx* ctx, double* total_ms, int* launches, int reset);

/*
 * gf_launch_count — number of CUDA kernels this context has enqueued since the last call with
 * reset != 0 (half-sweeps, reductions, reunitarisation, layout conversion, finalisation); memcpys are
 * not counted.  bench.py reports it as "gpu_launches".
 */
int gf_launch_count(gf_ctx* ctx, int64_t* launches, int reset);

/* bytes of device memory held by the context */
int64_t gf_device_bytes(const gf_ctx* ctx);

/* number of lattice sites V = Nx*Ny*Nz*Nt of the context (a links buffer holds V*4*18 reals, a transform V*18) */
int64_t gf_volume(const gf_ctx* ctx);

const char* gf_last_error(const gf_ctx* ctx);
const char* gf_version(void);

/*
 * Tuning hooks — NOT part of the contract (bench.py's side studies and two tests use them; results never depend on them
 * beyond what is said here).
 *   gf_debug_set_fused(ctx, 0)  gf_run measures with the stand-alone reduction kernels at every check instead of the
 *                               partial sums fused into the half-sweeps; same decisions, same results.
 *   gf_debug_set_pdl(ctx, 0)    half-sweeps are launched without programmatic dependent launch.
 *   gf_debug_set_block(ctx, n)  CTA size of the half-sweep kernel: a multiple of 32, capped at the kernel's maximum (128
 *                               threads for float storage, 64 for double and for the float stochastic rules); 0 = the
 *                               default, which is that maximum, or 32 where the whole lattice's half-sweep would not
 *                               give every SM a CTA.  Links are bit-identical for every n, fused partial sums differ in
 *                               summation order.
 */
int gf_debug_set_fused(gf_ctx* ctx, int fused);
int gf_debug_set_pdl(gf_ctx* ctx, int pdl);
int gf_debug_set_block(gf_ctx* ctx, int block);

#ifdef __cplusplus
}
#endif
#endif /* GF_H_ */
