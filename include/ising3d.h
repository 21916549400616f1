/*
 * ising3d.h -- C ABI of the B200-native zero-temperature coarsening sweep
 * of the periodic simple-cubic d=3 Ising model (arXiv 2305.12161).
 *
 * Citations are PAPER.md:<line> = /root/reference/PAPER.md; "D<n>" are the
 * readings listed in DESIGN.md section 3 for everything
 * the paper leaves open.
 *
 * The method (what every call below computes)
 * -------------------------------------------
 *  - Lattice: s(x,y,z) in {-1,+1}, 0 <= x,y,z < L, periodic in all three
 *    directions, nearest-neighbour coupling J = 1.
 *  - Start: iid +-1 spins with p = 1/2, i.e. T = infinity, m ~ 0.
 *  - Site rule, T -> 0 Glauber acceptance, eq. (6) PAPER.md:105-108:
 *    Delta E = 2 s_i sum_nn s_j;  flip if Delta E < 0, keep if Delta E > 0,
 *    flip with probability 1/2 if Delta E = 0 (here: iff the site's Philox bit
 *    is 1, D2/D5).
 *  - Sweep = checkerboard "01 cycle": all sites with
 *    (x+y+z) even ("black", colour 0) concurrently, then all sites with
 *    (x+y+z) odd ("white", colour 1), which see the updated black sites.
 *    One sweep = N = L^3 proposals = 1 MCS.
 *  - Measurements: N_up, the antiparallel-pair counts A_mu(r) along the three
 *    axes for r = 0..L/2 (eq. (2) PAPER.md:43 reduced to integers, D8), the
 *    number of broken nearest-neighbour bonds (interface energy
 *    E = -3N + 2 n_broken), the axis-averaged C(r,t) and ell(t) from
 *    C(ell,t) = c, c = 0.5 (D9).
 *
 * Canonical packed state (D3) -- the format of get_state / set_state
 * -------------------------------------------------------------------
 *  colour c = (x+y+z) mod 2.  Inside row (y,z) the colour-c sites are
 *  x = 2k + o, o = (y+z+c) mod 2, k = x>>1 = 0..L/2-1.  Bit index inside
 *  colour c: b = (z*L + y)*(L/2) + k; 32-bit word w = b>>5, bit j = b&31
 *  (LSB = smallest k); bit value 1 <=> s = +1.  One replica = colour-0 words
 *  (L^3/64 of them) followed by colour-1 words; replicas follow one another.
 *  Words per replica: L^3/32.
 *
 * Random bits (D5)
 * ----------------
 *  Philox4x32-10, key = (seed & 0xFFFFFFFF, seed >> 32) (the replica's seed),
 *  counter = (q, t, c, tag): q = b>>7 the 128-spin group inside the colour,
 *  t = 0-based index of the sweep being executed, c = colour being updated,
 *  tag = 0 for tie bits, 1 for the initial configuration (with t = 0).
 *  Output word i (0..3) bit j belongs to the spin at bit index 128q + 32i + j.
 *  Counter based: results never depend on thread order or launch shape.
 *
 * General conventions
 * -------------------
 *  - Every function returns ISING3D_OK (0) or a negative error code; no
 *    exception or abort crosses this boundary.  ising3d_last_error() gives a
 *    thread-local, never-NULL description of the last failure.
 *  - "host" / "device" is stated for every pointer.  The library owns all
 *    device memory it allocates and frees it in ising3d_free().
 *  - Handles are not thread safe; distinct handles are independent.
 *  - There is no CPU fallback: without a CUDA device every compute call
 *    fails with ISING3D_ECUDA.
 *  - L must be a multiple of 64 with 64 <= L <= 4096; 1 <= n_rep.
 */
#ifndef ISING3D_H_
#define ISING3D_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ISING3D_OK      0
#define ISING3D_EINVAL (-1)   /* bad argument (null pointer, bad L, n_rep, buffer too small,
                                 sweep counter would pass 2^32-1)                        */
#define ISING3D_ENOMEM (-2)   /* device or host allocation failed                         */
#define ISING3D_ECUDA  (-3)   /* CUDA runtime error; text in ising3d_last_error()         */

/* sweep-kernel variants (ising3d_set_variant) */
#define ISING3D_VARIANT_AUTO    0   /* resident (L <= 256), fused2 (L in 512..4096; switches to the
                                       activity-driven kernel when few groups can still change,
                                       see ising3d_set_activity_policy), else generic           */
#define ISING3D_VARIANT_GENERIC 1   /* two in-place half-sweep launches per sweep         */
#define ISING3D_VARIANT_FUSED   2   /* one launch per sweep, black+white fused            */
#define ISING3D_VARIANT_FUSED2  3   /* fused, two rows per thread (L in {512,1024,1536,2048,4096}); a batch
                                       is swept replica by replica (n_rep launches per sweep) */
#define ISING3D_VARIANT_RESIDENT 4  /* lattice resident in the shared memory of a thread-block
                                       cluster, all sweeps of a call in one launch (L in 64..256) */
#define ISING3D_VARIANT_FUSED3  5   /* two sweeps per launch, the state in between stays in shared
                                       memory (L in {1024, 2048}, 01 cycle); an odd last sweep and
                                       the mixed cycle run on fused2                           */

#define ISING3D_VARIANT_ACTIVE  6   /* activity-driven: only the 128-spin groups that hold a site with
                                       Delta E <= 0, or that read a word changed since their last
                                       evaluation, are evaluated (two launches per sweep, in place;
                                       L in {256,512,1024,2048,4096}, plain checkerboard, T = 0).
                                       Same trajectory; pays once few groups can change        */

/* measurement kernels (ising3d_set_measure_variant) */
#define ISING3D_MEASURE_AUTO     0  /* tensor where the shape allows (L % 512 == 0), else popcount */
#define ISING3D_MEASURE_POPCOUNT 1  /* XOR + carry-save popcount over line words, any L             */
#define ISING3D_MEASURE_TENSOR   2  /* pair counts as diagonals of a Gram matrix: tcgen05 int8 MMA  */

/* update order inside a sweep (ising3d_set_cycle) */
#define ISING3D_CYCLE_01    0   /* colour 0 then colour 1, every sweep (main text) */
#define ISING3D_CYCLE_MIXED 1   /* first colour drawn per sweep (Supp. I.B PAPER.md:258, D10)    */
#define ISING3D_CYCLE_DOUBLE_CB 2 /* double checkerboard, 01 cycle (Supp. I.A PAPER.md:223-240, D14) */
#define ISING3D_CYCLE_DOUBLE_CB_MIXED 3 /* double checkerboard, mixed cycle (Supp. I.B PAPER.md:258, D15) */

typedef struct ising3d ising3d_t;   /* opaque */

/*
 * Measurement record.  All arrays are HOST memory allocated by the CALLER;
 * the caller sets L, n_rep (must match the handle), c_intercept and the
 * pointers; ising3d_measure fills sweep and the arrays.
 */
typedef struct {
    int32_t   L, n_rep;
    uint64_t  sweep;        /* out: completed sweeps at the time of measurement           */
    uint64_t *n_up;         /* [n_rep]              number of +1 spins (D8)               */
    uint64_t *n_broken;     /* [n_rep]              antiparallel n.n. bonds = sum_mu A_mu(1) */
    uint64_t *antipar;      /* [n_rep][3][L/2+1]    A_mu(r), mu = x,y,z; A_mu(0) = 0      */
    double   *C;            /* [n_rep][L/2+1] or NULL   eq. (2), axis-averaged, fp64 (D9) */
    double   *ell;          /* [n_rep] or NULL          first C = c crossing, NaN if none */
    double    c_intercept;  /* 0.5 in the paper; other values: Table II     */
} ising3d_meas_t;

/* Device bytes needed by a handle with caller-provided memory
 * (ising3d_init_batch_with_buffer).  0 if L / n_rep are invalid. */
size_t ising3d_required_bytes(int L, int n_rep);

/* Number of 32-bit words of the canonical packed state of ONE replica: L^3/32. */
size_t ising3d_words_per_replica(int L);

/*
 * Create one lattice in the T = infinity start of `seed` (D6), sweep = 0.
 * PAPER.md:45.  *h is written only on success.  Runs on the legacy default
 * stream until ising3d_set_stream is called; the handle is created on the
 * CUDA device current at the time of the call, and every later call on it
 * must be made with that device current (handles on several devices may
 * live in one process).
 */
int ising3d_init(ising3d_t **h, int L, uint64_t seed);

/*
 * n_rep independent lattices ("independent realizations"),
 * replica i seeded with seeds[i] (HOST array of n_rep entries, copied).
 * All replicas advance in the same launches.  Replica i is bit-identical to
 * a single-lattice handle created with seeds[i].
 */
int ising3d_init_batch(ising3d_t **h, int L, int n_rep, const uint64_t *seeds);

/*
 * Same, in caller-provided DEVICE memory (e.g. a torch tensor): `dev_buf`
 * must be 256-byte aligned and hold >= ising3d_required_bytes(L, n_rep);
 * it stays owned by the caller and must outlive the handle.  `cuda_stream`
 * is a cudaStream_t (may be NULL = legacy default stream); the initial state
 * is generated on that stream.
 */
int ising3d_init_batch_with_buffer(ising3d_t **h, int L, int n_rep, const uint64_t *seeds,
                                   void *dev_buf, size_t dev_bytes, void *cuda_stream);

/* Re-generate the T = infinity start (same seeds) and reset sweep to 0. Async. */
int ising3d_reset(ising3d_t *h);

/* Choose the kernels behind the A_mu(r) counts of ising3d_measure (ISING3D_MEASURE_*).  Both
 * give the same integers (D8).  EINVAL if the shape does not support the requested variant. */
int ising3d_set_measure_variant(ising3d_t *h, int variant);

/*
 * Menger-sponge start (Fig. 4; reading D11): "The starting
 * configuration of dimensions L^3 is created by repeating sponges of k-th iteration of size
 * (3^k)^3.  For each sponge we pick uniformly at random whether the Menger structure is
 * represented by up or down spins."  Tiles start at the origin, the last tile in each
 * direction is cut at L; a site with local coordinates (u,v,w) is in the sponge iff at no
 * ternary digit position two or more of u,v,w have digit 1; tile T = (Z*nT + Y)*nT + X,
 * nT = ceil(L/3^k), takes its sign from bit (T & 127) of Philox(key = the replica's seed,
 * counter = (T >> 7, k, 0, 3)): sponge sites +1 if the bit is 1, holes the opposite sign.
 * k = 0 is an iid p = 1/2 start.  Replaces the state of every replica, sets sweep to 0.
 * Asynchronous.  EINVAL unless 0 <= k <= 7 and 3^k <= L.
 */
int ising3d_init_menger(ising3d_t *h, int k);

/*
 * Choose the order of the two half-sweeps (ISING3D_CYCLE_*).  01 cycle (default): colour 0
 * then colour 1 (D7).  Mixed cycle (Supp. I.B PAPER.md:258: "choosing at random
 * which sublattice to update first ... still every spin is proposed to flip exactly once per
 * sweep"; reading D10): in sweep t the replica with seed s updates first the colour given by
 * bit 0 of word 0 of Philox(key = s, counter = (0, t, 0, 2)); the tie bits keep counter
 * (q, t, c, 0) with c the colour being updated.  Double checkerboard (Supp. I.A PAPER.md:223-240;
 * reading D14): cubic blocks of edge 8 starting at the origin form a coarse checkerboard
 * (coarse colour (x/8 + y/8 + z/8) mod 2); a sweep updates the red blocks (their darker sites,
 * (x+y+z) even, then their lighter sites) with everything else frozen, then the blue blocks:
 * four masked half-sweeps, every spin proposed once, tie bits as in the plain checkerboard.
 * Runs on the resident (L <= 256), fused2 (L in 512..4096: one masked launch per coarse colour,
 * dark then light sites inside it) and generic kernels.  Its mixed cycle (Table I;
 * reading D15): the coarse colour updated first in sweep t is the D10 bit; block
 * Bi = (bz*nB + by)*nB + bx (nB = L/8) updates first the fine colour given by bit (Bi & 127) of
 * Philox(key = seed, counter = (Bi >> 7, t, 0, 36)), then the other; fused2 (L in 512..4096: the
 * block bits of a sweep are drawn into a bit array, then per coarse colour one masked launch for
 * the blocks that drew "dark first" and one for those that drew "light first") and generic
 * kernels.  Takes effect from the next sweep.
 * EINVAL for an unknown value, with ISING3D_VARIANT_FUSED (01 cycle only), for the double
 * checkerboard with ISING3D_VARIANT_FUSED3 or _ACTIVE, or at T > 0 for anything but the 01 cycle.
 */
int ising3d_set_cycle(ising3d_t *h, int cycle);

/*
 * Temperature of the quench.  T = 0 (default): the paper's T -> 0 acceptance, eq. (6)
 * PAPER.md:105-108 ("which is the acceptance probability we use throughout").  T > 0 (k_B = 1):
 * the Glauber probability of eq. (5), p = 1 / (1 + exp(Delta E / T)) (the paper's
 * announced follow-up).  Reading D13: a site with n antiparallel
 * neighbours (Delta E = 12 - 4n) flips iff u < thr[n], thr[n] = floor(2^32 p) in [0, 2^32]
 * (fp64), u = sum_j b_j 2^(31-j) its 32-bit uniform of the sweep, b_j the site's bit of
 * Philox(key = seed, counter = (q, t, c, 4 + j)), j = 0..31.  Sweeps at T > 0 run the
 * "glauber" kernel (two launches per sweep, any L, batches) whatever the sweep variant.
 * EINVAL for negative or non-finite T.
 */
int ising3d_set_temperature(ising3d_t *h, double T);

/* Use `cuda_stream` (a cudaStream_t owned by the caller) for all later work. */
int ising3d_set_stream(ising3d_t *h, void *cuda_stream);

/* Choose the sweep kernel (ISING3D_VARIANT_*).  EINVAL if the shape does not
 * support the requested variant.  All variants give bit-identical states. */
int ising3d_set_variant(ising3d_t *h, int variant);

/*
 * Activity of the state (eq. (6): a site can change only if Delta E <= 0, i.e.
 * n >= 3 of its six neighbours are antiparallel).  awake_groups: HOST [n_rep][2] or NULL; entry
 * [rep][c] = number of 128-spin groups (the Philox groups q of D5) of colour c that hold at least
 * one site with n >= 3 in the current state -- an exact integer, a function of the state only.
 * last_fraction: HOST or NULL; with awake_groups the fraction of such groups (both colours, all
 * replicas), without it the fraction seen by the last probe of the AUTO policy (-1 if none yet).
 * Counting needs L in {256,512,1024,2048,4096} (EINVAL otherwise) and synchronises the stream.
 */
int ising3d_activity(ising3d_t *h, uint64_t *awake_groups, double *last_fraction);

/*
 * Work done by the activity-driven kernel since the last call (or since the handle was created):
 * evaluated_changed HOST [n_rep][2] = 128-spin groups evaluated (both colours, all sweeps) and
 * groups whose words changed.  A diagnostic of the kernel, not of the state: evaluated groups are
 * the ones holding a Delta E <= 0 site plus the ones woken by a neighbour's change.  Resets the
 * tallies; synchronises the stream.  EINVAL unless L in {256,512,1024,2048,4096}.
 */
int ising3d_active_stats(ising3d_t *h, uint64_t *evaluated_changed);

/*
 * Policy of ISING3D_VARIANT_AUTO at L >= 512 (T = 0, plain checkerboard): after every
 * `probe_interval` dense sweeps the activity flags are rebuilt and counted on the stream; once the
 * fraction of groups that can change has been seen below `on_below`, the following sweeps run on
 * the activity-driven kernel.  That kernel tallies the groups it finds holding a Delta E <= 0 site;
 * every probe_interval sweeps the tally is read, and if its mean per colour update passes
 * `off_above` (as a fraction of the groups of a colour) the handle goes back to fused2.
 * No probe blocks the host: the counts go to pinned memory, an event marks them, and the library
 * looks at the event (cudaEventQuery) between launches and at the start of the next ising3d_sweep
 * call, so a switch takes effect some sweeps after the probe that caused it -- at most one probe is
 * in flight, and one that the GPU has not reached yet makes the next one be skipped.  The choice
 * changes the speed only, never the result.  probe_interval = 0: always fused2.  Defaults: 1024,
 * 0.11, 0.14 (measured break-even of the two kernels at L = 2048).  Changing the
 * temperature, the cycle, the variant, the policy or the state puts the handle back on fused2.
 * EINVAL unless 0 <= on_below <= off_above <= 1.
 */
int ising3d_set_activity_policy(ising3d_t *h, uint64_t probe_interval, double on_below, double off_above);

/*
 * Thread-block cluster size of the resident kernel (L in {64,128,256}): the lattice is split
 * into `cs` z slabs, one CTA (= one SM) each, halo planes exchanged through distributed shared
 * memory after every half-sweep.  cs = 0 restores the automatic choice (the
 * smallest cluster whose slab fits shared memory, grown while all replicas stay co-resident).
 * The result does not depend on cs.  EINVAL unless cs is a power of two <= 16 with L/cs >= 2
 * whose slab fits 200 KB of shared memory and that the device can schedule, or for other L.
 */
int ising3d_set_cluster_size(ising3d_t *h, int cs);

/*
 * Run n_sweeps checkerboard sweeps (eq. (6)).
 * Asynchronous on the handle's stream; no host synchronisation inside, under every variant
 * and policy (the AUTO policy's probes are queued on the stream and read back through pinned
 * memory and an event, ising3d_set_activity_policy).  Inside a stream capture the call records
 * sweeps only, on the kernel the handle was dispatching when the capture began.
 * The sweep counter advances by n_sweeps; EINVAL if it would pass 2^32-1.
 */
int ising3d_sweep(ising3d_t *h, uint64_t n_sweeps);

/*
 * Integer measurements + fp64 post-processing (D8, D9; eq. (2) PAPER.md:43,
 * ell from C = c PAPER.md:51).  Synchronises the handle's stream.  Does not
 * change the state or the sweep counter.  The tensor-core variant uses the
 * handle's second (ping-pong) state buffer as scratch; that buffer never holds
 * live data between calls.
 */
int ising3d_measure(ising3d_t *h, ising3d_meas_t *out);

/*
 * ising3d_measure_static -- N_up and A_mu(r) of a packed state the caller already holds on the
 * device, for callers that must not allocate device memory.
 *
 * Who this is for.  Every other entry point works on a handle, and creating a handle either
 * calls cudaMalloc or asks the caller to bring a buffer of ising3d_required_bytes().  Some users
 * of this library can do neither at the point where they want a measurement:
 *  - code that runs inside a service whose device memory is handed out once at start-up by a
 *    pool it does not control (a framework's caching allocator that has already taken the whole
 *    GPU, a job scheduler with a fixed per-tenant budget): a cudaMalloc there fails, or succeeds
 *    and breaks the budget somebody else relies on;
 *  - code on a latency-critical path (an analysis hook called between sweeps of a running
 *    simulation, a monitoring thread): cudaMalloc and cudaFree serialise against all work on the
 *    device, so one measurement would stall every other stream;
 *  - code that only has the spins, e.g. a state produced by another program in the D3 format,
 *    and wants the counts without building a simulation handle around them.
 * For them the accumulators the measurement kernels add into live in a fixed array that is part
 * of the library image itself (a file-scope __device__ array in ising3d.cu).  Nothing is
 * allocated or freed by this call, by the library on its behalf, or by any routine it uses;
 * cuFFT and the tensor-core path (which borrows a lattice-sized buffer) are not involved: the
 * counts come from the XOR + carry-save popcount kernels (ISING3D_MEASURE_POPCOUNT), which give
 * the same integers (D8; eq. (2) PAPER.md:43 reduced to counts).
 *
 *   dev_words  DEVICE  in   n_rep * L^3/32 words, canonical packed state D3 (the get_state
 *                           format), 16-byte aligned; read only, owned by the caller
 *   n_up       HOST    out  [n_rep]            number of +1 spins
 *   antipar    HOST    out  [n_rep][3][L/2+1]  A_mu(r), mu = x,y,z; A_mu(0) = 0
 *   cuda_stream             a cudaStream_t (NULL = legacy default stream); the call queues its work
 *                           there and waits for that stream before returning
 * n_broken, C(r) and ell are plain host arithmetic on these integers (see ising3d_meas_t and D9).
 *
 * The limit.  The array holds ISING3D_STATIC_MAX_COUNTS 64-bit counters (128 KiB; every GPU that
 * loads the library carries it until the process ends).  A call needs n_rep * (1 + 3 (L/2+1)) of
 * them: one lattice of any supported L (L = 4096 needs 6 148), 64 replicas of L = 128, 42 of
 * L = 256.  A larger request is refused with ISING3D_EINVAL and a message that names both numbers;
 * split the batch over several calls (dev_words + k * L^3/32 is replica k).
 *
 * First call on a device.  It looks up the device address of the array (cudaGetSymbolAddress)
 * and raises the kernels' shared-memory limit, once per device and process, with the device
 * that is current at the call.  Make that first call during set-up, before any stream capture
 * is begun.  Later calls on that device only launch kernels and copy the results.
 *
 * Sharing.  All calls on one GPU, from any thread, use the same array, and it keeps whatever
 * the previous call left there.  The call clears the part it uses before counting, so results
 * never depend on earlier calls; but two calls whose GPU work overlaps (different streams, or
 * different threads) add into the same counters and both return garbage.  Run them one after
 * the other.  Handles and ising3d_measure are unaffected: they never touch this array.
 */
#define ISING3D_STATIC_MAX_COUNTS 16384
int ising3d_measure_static(const uint32_t *dev_words, int L, int n_rep, uint64_t *n_up, uint64_t *antipar,
                           void *cuda_stream);

/*
 * The paper's own estimator: the full correlation matrix by eq. (7)
 * PAPER.md:128, mean_i s_i s_{i+k} = [F^-1(|F s|^2)]_k (3-D real-data DFT in place, fp64, cuFFT),
 * then "radially averaging over the three-dimensional correlation matrix", and
 * the structure factor S(k) = |F s|^2 / N.  Reading D12: displacements are folded to
 * the minimal image (components in (-L/2, L/2]) and binned by the integer nearest to |d|
 * ((2b-1)^2 <= 4|d|^2 < (2b+1)^2), bins b = 0..L/2; the same bins in index space for k.
 * The transform of +-1 data is an integer up to round-off, so P(d) = sum_i s_i s_{i+d} is
 * recovered exactly (llrint) and corr_sum holds exact integer sums.
 *   corr_sum [n_rep][L/2+1]  HOST  sum of P(d) over bin b
 *   shell    [L/2+1]         HOST  number of displacements in bin b
 *   C_rad    [n_rep][L/2+1]  HOST  corr_sum / (N * shell) - m^2            (eq. 2)
 *   S_rad    [n_rep][L/2+1]  HOST  may be NULL; mean of |F s|^2 / N over the k bin
 *   ell      [n_rep]         HOST  may be NULL; first C_rad = c_intercept crossing (D9 rule)
 * Needs 8 bytes per site of device memory plus the cuFFT work area, allocated by the library
 * on first use (ENOMEM if that fails; the handle stays usable).  Synchronises the stream.
 */
typedef struct {
    int32_t   L, n_rep;
    uint64_t  sweep;
    int64_t  *corr_sum;
    uint64_t *shell;
    double   *C_rad;
    double   *S_rad;
    double   *ell;
    double    c_intercept;
} ising3d_radial_t;
int ising3d_measure_radial(ising3d_t *h, ising3d_radial_t *out);

/* Exactness margin of the last ising3d_measure_radial call (D12): the largest distance of an
 * inverse-transform value / N from the integer it was rounded to, over all displacements and
 * replicas; P(d) is exact as long as this stays below 1/2 (it is of order 1e-4 at L = 2048).
 * HOST pointer; -1 before the first call. */
int ising3d_radial_rounding(const ising3d_t *h, double *max_distance);

/* Give back the device memory and cuFFT plans ising3d_measure_radial keeps between calls
 * (8 bytes per site + work area: 128 GiB at L = 2048).  The next call re-creates them. */
int ising3d_release_radial(ising3d_t *h);

/*
 * Copy the canonical packed state (D3) to / from HOST memory.
 * n_words must equal n_rep * L^3/32.  Both synchronise the stream.
 * set_state also sets the sweep counter (the next sweep executed has index
 * `sweep`), which with the counter-based RNG resumes a run exactly.
 */
int ising3d_get_state(ising3d_t *h, uint32_t *words, size_t n_words, uint64_t *sweep);
int ising3d_set_state(ising3d_t *h, const uint32_t *words, size_t n_words, uint64_t sweep);

/* Same with DEVICE pointers (device-to-device copies on the handle's stream,
 * asynchronous).  Used to keep inputs resident in HBM.                        */
int ising3d_get_state_device(ising3d_t *h, uint32_t *dev_words, size_t n_words, uint64_t *sweep);
int ising3d_set_state_device(ising3d_t *h, const uint32_t *dev_words, size_t n_words, uint64_t sweep);

/* Introspection: shape, completed sweeps, kernels launched so far by this handle. */
int      ising3d_L(const ising3d_t *h);
int      ising3d_n_rep(const ising3d_t *h);
uint64_t ising3d_sweep_count(const ising3d_t *h);
uint64_t ising3d_launch_count(const ising3d_t *h);
/* name of the sweep kernel the handle currently dispatches to ("generic", "fused", ...) */
const char *ising3d_variant_name(const ising3d_t *h);
/* "tensor" or "popcount": the measurement kernels the handle dispatches to */
const char *ising3d_measure_variant_name(const ising3d_t *h);
/* CTAs per thread-block cluster (= SMs per lattice) of the resident kernel; 0 if another
 * kernel is dispatched. */
int ising3d_cluster_size(const ising3d_t *h);

/* Block until all work queued on the handle's stream is done.  A probe of the AUTO policy that
 * was in flight has landed by then and its result is applied (so has it after ising3d_get_state):
 * ising3d_variant_name and ising3d_activity's last_fraction are up to date afterwards. */
int ising3d_sync(ising3d_t *h);

/* Release the handle and all memory the library allocated for it. NULL is a no-op. */
void ising3d_free(ising3d_t *h);

/* Thread-local description of the last error on this thread; never NULL. */
const char *ising3d_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ISING3D_H_ */
