/*
 * oracle/ising_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, site-by-site CPU statement of what the hot path of
 * arXiv 2305.12161 computes: the zero-temperature single-spin-flip
 * checkerboard sweep of the periodic simple-cubic d=3 Ising model and the
 * integer measurements behind energy, magnetisation and C(r,t).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may build, load or call this file.  It shares no code,
 * header, table or constant generator with paper_2305_12161_b200/csrc (the
 * CUDA path); the two meet only in the tests, which compare their outputs.
 *
 * One int8 per spin, literal Delta-E rule, literal modular neighbour indexing.
 * No blocking, no bit tricks, no fusion: every function is meant to be checked
 * against the cited passage by eye.
 *
 * Citations are PAPER.md:<line> and SURVEY.md
 * section 8(c) definitions D1..D9 (the readings taken where the paper is
 * silent; they are listed again in DESIGN.md).
 *
 * Pins (tests/test_oracle_*.py, all run with -m "not gpu"):
 *   orc_philox4x32_10   : known-answer vectors, NVIDIA's curand host path,
 *                         big-integer Python restatement
 *   orc_half_sweep      : exhaustive 2^6 x 2 x 2 site table, brute-force
 *                         H(flipped)-H(config) variant on L=4,6,8, closed
 *                         forms (Neel state, single spin, 2x2x2 cube), fixed
 *                         points, order independence, energy monotonicity
 *   orc_init_random     : bit statistics, independent Python restatement
 *   orc_measure         : closed forms (slab, all-up), translation and axis
 *                         permutation invariance, numpy restatement
 *   orc_postprocess     : closed forms, hand-worked example
 *   orc_export/import   : round trip, independent Python packer
 *   orc_site_after      : equals orc_sweep site by site on small L
 *   orc_activity        : all up -> 0, Neel -> all groups, one reversed spin -> one group,
 *                         equals "some tie-bit assignment changes the group" by brute force
 *   orc_first_colour / orc_sweep_mixed : Neel state closed form (the first colour
 *                         decides the sign of the ordered state), bit statistics,
 *                         big-integer Python Philox
 *   orc_menger_solid / orc_init_menger / orc_menger_site : solid counts 20^k, the k = 1 cross
 *                         written out, self-similarity, tile-sign statistics, k = 0 iid; the
 *                         single-site form equals the array form site by site and the big-integer
 *                         Python Philox on tiles beyond 2^32
 *   orc_corr_direct / orc_radial_bin / orc_radial_sums : P(0) = N, sum_d P(d) = M^2,
 *                         P along the axes = N - 2 A_mu(r) (orc_measure), slab closed form,
 *                         shell counts against a set-based Python count, bins vs exact
 *                         rational comparison
 *   orc_half_sweep_dcb / orc_sweep_dcb : B = L reduces to the plain 01 sweep, pure-Python
 *                         restatement on L = 8, every site proposed once (Neel read-out per
 *                         block colour), fixed points, energy monotone
 *   orc_block_first_fine / orc_sweep_dcb_mixed : documented Philox bits, Neel read-out of the
 *                         coarse order and of every block's fine order, pure-Python restatement,
 *                         every site proposed once, energy monotone
 *   orc_glauber_thresholds / orc_site_uniform / orc_sweep_T : p(6-n) = 1 - p(n), p(3) = 1/2,
 *                         hand-computed thresholds, T -> infinity closed form (flip iff the top
 *                         Philox plane bit is 0), acceptance frequencies on uniform-n states
 *                         (all up: n = 0, Neel: n = 6) within binomial errors, T -> 0 limit of
 *                         the deterministic moves, energy relaxation towards the T = 0 quench
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ */
/* D5: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).              */
/* counter (c0,c1,c2,c3), key (k0,k1), all uint32.                     */
/* One round: p0 = M0*c0, p1 = M1*c2 (64-bit products);                */
/*   new counter = (hi(p1)^c1^k0, lo(p1), hi(p0)^c3^k1, lo(p0)).       */
/* Ten rounds; the key is bumped by (W0,W1) between rounds (9 times).  */
/* ------------------------------------------------------------------ */
#define ORC_PHILOX_M0 0xD2511F53u
#define ORC_PHILOX_M1 0xCD9E8D57u
#define ORC_PHILOX_W0 0x9E3779B9u
#define ORC_PHILOX_W1 0xBB67AE85u

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += ORC_PHILOX_W0;
            k1 += ORC_PHILOX_W1;
        }
        uint64_t p0 = (uint64_t)ORC_PHILOX_M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)ORC_PHILOX_M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------ */
/* The lattice: D1.  s[(z*L + y)*L + x] in {-1,+1}, periodic, L even.  */
/* ------------------------------------------------------------------ */
typedef struct {
    int      L;
    uint64_t seed;
    uint32_t sweep;      /* completed sweeps (MCS) */
    int8_t  *s;
} orc_t;

static inline size_t orc_idx(const orc_t *o, int x, int y, int z)
{
    return ((size_t)z * (size_t)o->L + (size_t)y) * (size_t)o->L + (size_t)x;
}

/* a mod L for -L <= a < 2L (all that periodic neighbours and r <= L/2 need) */
static inline int orc_mod(int a, int L)
{
    if (a >= L) return a - L;
    if (a < 0)  return a + L;
    return a;
}

orc_t *orc_create(int L, uint64_t seed)
{
    if (L < 4 || (L & 1)) return NULL;
    orc_t *o = (orc_t *)calloc(1, sizeof(orc_t));
    if (!o) return NULL;
    o->L = L;
    o->seed = seed;
    o->sweep = 0;
    o->s = (int8_t *)malloc((size_t)L * L * L);
    if (!o->s) { free(o); return NULL; }
    memset(o->s, 1, (size_t)L * L * L);   /* all up until initialised */
    return o;
}

void orc_free(orc_t *o)
{
    if (!o) return;
    free(o->s);
    free(o);
}

int8_t  *orc_spins(orc_t *o)            { return o->s; }
uint32_t orc_get_sweep(const orc_t *o)  { return o->sweep; }
void     orc_set_sweep(orc_t *o, uint32_t t) { o->sweep = t; }
void     orc_set_seed(orc_t *o, uint64_t seed) { o->seed = seed; }

/* ------------------------------------------------------------------ */
/* D3: canonical packed position of a site.                            */
/*   colour c = (x+y+z) mod 2; k = x>>1;                               */
/*   bit index inside colour c: b = (z*L + y)*(L/2) + k;               */
/*   group q = b>>7, word-in-group i = (b>>5)&3, bit j = b&31.         */
/* ------------------------------------------------------------------ */
static inline uint64_t orc_bit_index(int L, int x, int y, int z)
{
    return ((uint64_t)z * (uint64_t)L + (uint64_t)y) * (uint64_t)(L / 2) + (uint64_t)(x >> 1);
}

/* D5 keying: key = (seed lo, seed hi); counter = (q, t, c, tag);
 * tag 0 = tie bits of sweep t, tag 1 = initial configuration (t = 0).
 * The site's bit is bit j of output word i.                            */
int orc_site_bit(uint64_t seed, int L, int x, int y, int z, uint32_t t, uint32_t tag)
{
    uint32_t c = (uint32_t)((x + y + z) & 1);
    uint64_t b = orc_bit_index(L, x, y, z);
    uint32_t ctr[4] = { (uint32_t)(b >> 7), t, c, tag };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    return (int)((out[(b >> 5) & 3] >> (b & 31)) & 1u);
}

/* D6 ("random spin configurations (with magnetization m ~ 0)"):
 * spin = +1 iff its Philox(tag=1, t=0) bit is 1.                       */
void orc_init_random(orc_t *o)
{
    const int L = o->L;
    #pragma omp parallel for schedule(static)
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x)
                o->s[orc_idx(o, x, y, z)] =
                    orc_site_bit(o->seed, L, x, y, z, 0u, 1u) ? (int8_t)1 : (int8_t)-1;
    o->sweep = 0;
}

/* ------------------------------------------------------------------ */
/* D2: the T -> 0 Glauber rule, eq. (6):              */
/*   Delta E < 0 : accept;  Delta E > 0 : reject;                      */
/*   Delta E = 0 : accept with probability 1/2 (here: iff the site's   */
/*   random bit is 1).  H = -sum_<ij> s_i s_j, so flipping s_i changes */
/*   the energy by Delta E = 2 s_i sum_{j in nn(i)} s_j. */
/* ------------------------------------------------------------------ */
static inline void orc_update_site(orc_t *o, int x, int y, int z, uint32_t t)
{
    const int L = o->L;
    int h = o->s[orc_idx(o, orc_mod(x + 1, L), y, z)]
          + o->s[orc_idx(o, orc_mod(x - 1, L), y, z)]
          + o->s[orc_idx(o, x, orc_mod(y + 1, L), z)]
          + o->s[orc_idx(o, x, orc_mod(y - 1, L), z)]
          + o->s[orc_idx(o, x, y, orc_mod(z + 1, L))]
          + o->s[orc_idx(o, x, y, orc_mod(z - 1, L))];
    int8_t *si = &o->s[orc_idx(o, x, y, z)];
    int dE = 2 * (int)(*si) * h;
    if (dE < 0) {
        *si = (int8_t)(-*si);
    } else if (dE == 0) {
        if (orc_site_bit(o->seed, L, x, y, z, t, 0u)) *si = (int8_t)(-*si);
    }
}

/* D7 half-sweep: every site of colour c = (x+y+z) mod 2 is
 * proposed exactly once; neighbours all have the other colour and are frozen.
 * order: 0 = lexicographic (z,y,x), 1 = reverse lexicographic,
 *        2 = a seeded random permutation of the sites (small L; pin P6).   */
void orc_half_sweep(orc_t *o, uint32_t t, int c, int order, uint64_t order_seed)
{
    const int L = o->L;
    if (order == 0) {
        /* same-colour sites do not interact, so planes can go
         * in parallel without changing any result (checked by pin P6). */
        #pragma omp parallel for schedule(static)
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x)
                    if (((x + y + z) & 1) == c) orc_update_site(o, x, y, z, t);
    } else if (order == 1) {
        for (int z = L - 1; z >= 0; --z)
            for (int y = L - 1; y >= 0; --y)
                for (int x = L - 1; x >= 0; --x)
                    if (((x + y + z) & 1) == c) orc_update_site(o, x, y, z, t);
    } else {
        size_t N = (size_t)L * L * L;
        uint32_t *perm = (uint32_t *)malloc(N * sizeof(uint32_t));
        for (size_t i = 0; i < N; ++i) perm[i] = (uint32_t)i;
        uint64_t st = order_seed * 6364136223846793005ull + 1442695040888963407ull;
        for (size_t i = N - 1; i > 0; --i) {           /* Fisher-Yates */
            st = st * 6364136223846793005ull + 1442695040888963407ull;
            size_t j = (size_t)((st >> 33) % (uint64_t)(i + 1));
            uint32_t tmp = perm[i]; perm[i] = perm[j]; perm[j] = tmp;
        }
        for (size_t i = 0; i < N; ++i) {
            int x = (int)(perm[i] % (uint32_t)L);
            int y = (int)((perm[i] / (uint32_t)L) % (uint32_t)L);
            int z = (int)(perm[i] / ((uint32_t)L * (uint32_t)L));
            if (((x + y + z) & 1) == c) orc_update_site(o, x, y, z, t);
        }
        free(perm);
    }
}

/* D7 sweep = "01 cycle": colour 0 fully, then colour 1
 * (which sees the updated colour 0).  One sweep = N proposals = 1 MCS.     */
void orc_sweep(orc_t *o, uint64_t n_sweeps)
{
    for (uint64_t i = 0; i < n_sweeps; ++i) {
        orc_half_sweep(o, o->sweep, 0, 0, 0);
        orc_half_sweep(o, o->sweep, 1, 0, 0);
        o->sweep += 1;
    }
}

/* ------------------------------------------------------------------ */
/* Activity of a state (what ising3d_activity counts).  eq. (6)        */
/* PAPER.md:105-108 changes a site only if Delta E <= 0, Delta E =     */
/* 2 s_i sum_nn s_j.  out[c] = number of 128-spin groups */
/* q = b>>7 (D3/D5) of colour c that hold at least one site with       */
/* Delta E <= 0 in the current configuration.  A function of the       */
/* state only; no random numbers.                                      */
/* Pins: all up -> 0; Neel -> every group; one reversed spin -> 1      */
/* group of its colour, 0 of the other; a group counts iff a half-     */
/* sweep with some tie-bit assignment could change it (checked         */
/* against orc_half_sweep with both seeds' bits on small L).           */
/* ------------------------------------------------------------------ */
void orc_activity(const orc_t *o, uint64_t out[2])
{
    const int L = o->L;
    const uint64_t groups = ((uint64_t)L * L * (L / 2) + 127u) >> 7;   /* per colour */
    uint8_t *mark = (uint8_t *)calloc(2 * groups, 1);
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int h = o->s[orc_idx(o, orc_mod(x + 1, L), y, z)]
                      + o->s[orc_idx(o, orc_mod(x - 1, L), y, z)]
                      + o->s[orc_idx(o, x, orc_mod(y + 1, L), z)]
                      + o->s[orc_idx(o, x, orc_mod(y - 1, L), z)]
                      + o->s[orc_idx(o, x, y, orc_mod(z + 1, L))]
                      + o->s[orc_idx(o, x, y, orc_mod(z - 1, L))];
                int dE = 2 * (int)o->s[orc_idx(o, x, y, z)] * h;
                if (dE <= 0) {
                    int c = (x + y + z) & 1;
                    mark[(uint64_t)c * groups + (orc_bit_index(L, x, y, z) >> 7)] = 1;
                }
            }
    out[0] = out[1] = 0;
    for (uint64_t g = 0; g < groups; ++g) {
        out[0] += mark[g];
        out[1] += mark[groups + g];
    }
    free(mark);
}

/* ------------------------------------------------------------------ */
/* Mixed cycle (Supp. I.B PAPER.md:258): "choosing at */
/* random which sublattice to update first ... still every spin is      */
/* proposed to flip exactly once per sweep".  Reading D10: the first    */
/* colour of sweep t is bit 0 of word 0 of Philox(key = seed, counter = */
/* (0, t, 0, tag = 2)); the tie bits keep counter (q, t, c, 0) with c   */
/* the colour being updated.                                            */
/* ------------------------------------------------------------------ */
int orc_first_colour(uint64_t seed, uint32_t t)
{
    uint32_t ctr[4] = { 0u, t, 0u, 2u };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    return (int)(out[0] & 1u);
}

void orc_sweep_mixed(orc_t *o, uint64_t n_sweeps)
{
    for (uint64_t i = 0; i < n_sweeps; ++i) {
        int first = orc_first_colour(o->seed, o->sweep);
        orc_half_sweep(o, o->sweep, first, 0, 0);
        orc_half_sweep(o, o->sweep, 1 - first, 0, 0);
        o->sweep += 1;
    }
}

/* ------------------------------------------------------------------ */
/* Double-checkerboard update, 01 cycle (Supp. I.A    */
/* PAPER.md:223-240): the lattice is cut into cubic blocks forming a    */
/* coarse checkerboard; one sweep = kernel on the red blocks (update    */
/* the darker sites of each block, barrier, the lighter sites, write    */
/* back), then the same on the blue blocks.  While a coarse colour is   */
/* being updated its halo in the other blocks is frozen, so the sweep   */
/* is four masked half-sweeps: (coarse 0, fine 0), (coarse 0, fine 1),  */
/* (coarse 1, fine 0), (coarse 1, fine 1).  Reading D14: block edge B   */
/* (the paper gives none; the library uses B = 8), blocks start at the  */
/* origin, coarse colour = (x/B + y/B + z/B) mod 2 (L/B even), fine     */
/* colour = (x+y+z) mod 2 ("darker" = 0), red = coarse 0 first; tie bit */
/* of a site = its Philox bit with counter (q, t, fine colour, 0) as in */
/* the plain checkerboard: every site is proposed once per sweep.       */
/* ------------------------------------------------------------------ */
void orc_half_sweep_dcb(orc_t *o, uint32_t t, int coarse, int fine, int B)
{
    const int L = o->L;
    #pragma omp parallel for schedule(static)
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x)
                if (((x + y + z) & 1) == fine && ((x / B + y / B + z / B) & 1) == coarse)
                    orc_update_site(o, x, y, z, t);
}

void orc_sweep_dcb(orc_t *o, uint64_t n_sweeps, int B)
{
    for (uint64_t i = 0; i < n_sweeps; ++i) {
        for (int coarse = 0; coarse < 2; ++coarse)
            for (int fine = 0; fine < 2; ++fine)
                orc_half_sweep_dcb(o, o->sweep, coarse, fine, B);
        o->sweep += 1;
    }
}

/* ------------------------------------------------------------------ */
/* Double checkerboard, mixed cycle (Supp. I.B PAPER.md:258; Table I    */
/* "(mixed cycle) - double-checkerboard"): "the order of the coarse     */
/* checkerboards (red or blue first) is chosen at random once per sweep */
/* and the order of the fine checkerboard (lighter or darker sites      */
/* first) is chosen at random and independently for each (red or blue)  */
/* block and once per sweep."  Reading D15: the coarse colour updated   */
/* first in sweep t is orc_first_colour(seed, t) (the bit of D10); the  */
/* block with index Bi = (bz*nB + by)*nB + bx, nB = L/B, updates first  */
/* the fine colour given by bit (Bi & 127) of Philox(key = seed,        */
/* counter = (Bi >> 7, t, 0, tag 36)), then the other; tie bits as      */
/* before.  Each of the two kernels of a sweep is then two masked       */
/* passes: in every block of the coarse colour, first its first fine    */
/* colour, then (after the barrier of step 4/6) the   */
/* other.                                                               */
/* ------------------------------------------------------------------ */
int orc_block_first_fine(uint64_t seed, uint32_t t, uint32_t Bi)
{
    uint32_t ctr[4] = { Bi >> 7, t, 0u, 36u };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    return (int)((out[(Bi >> 5) & 3] >> (Bi & 31)) & 1u);
}

/* one pass: blocks of colour `coarse`; pass 0 updates each block's first fine colour, pass 1 the other */
void orc_pass_dcb_mixed(orc_t *o, uint32_t t, int coarse, int pass, int B)
{
    const int L = o->L, nB = L / B;
    #pragma omp parallel for schedule(static)
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int bx = x / B, by = y / B, bz = z / B;
                if (((bx + by + bz) & 1) != coarse) continue;
                uint32_t Bi = (uint32_t)((bz * nB + by) * nB + bx);
                int fine = orc_block_first_fine(o->seed, t, Bi) ^ pass;
                if (((x + y + z) & 1) == fine) orc_update_site(o, x, y, z, t);
            }
}

void orc_sweep_dcb_mixed(orc_t *o, uint64_t n_sweeps, int B)
{
    for (uint64_t i = 0; i < n_sweeps; ++i) {
        int first = orc_first_colour(o->seed, o->sweep);
        for (int k = 0; k < 2; ++k)
            for (int pass = 0; pass < 2; ++pass)
                orc_pass_dcb_mixed(o, o->sweep, k == 0 ? first : 1 - first, pass, B);
        o->sweep += 1;
    }
}

/* ------------------------------------------------------------------ */
/* Menger-sponge start: "The starting   */
/* configuration of dimensions L^3 is created by repeating sponges of   */
/* k-th iteration of size (3^k)^3.  For each sponge we pick uniformly   */
/* at random whether the Menger structure is represented by up or down  */
/* spins."  A site with local coordinates (u,v,w) in [0,3^k)^3 belongs  */
/* to the k-th iteration sponge iff at no ternary digit position two or */
/* more of u, v, w have the digit 1 (the removed cross of each 3x3x3).  */
/* Reading D11: tiles start at the origin, the last tile in each        */
/* direction is cut off at L (L need not be a multiple of 3^k, cf.      */
/* Fig. 4(b): 128^3 from 27^3 sponges); tile (X,Y,Z) has    */
/* linear index T = (Z*nT + Y)*nT + X, nT = ceil(L/3^k); its sign bit   */
/* is bit (T & 31) of word ((T >> 5) & 3) of Philox(key = seed, counter */
/* = (T >> 7, k, 0, tag = 3)); sponge sites get +1 if the bit is 1,     */
/* holes the opposite sign.  k = 0 gives one site per tile: an iid      */
/* p = 1/2 start ("k = 0 (corresponding to our case from    */
/* before)").                                                           */
/* ------------------------------------------------------------------ */
int orc_menger_solid(int u, int v, int w, int k)
{
    for (int level = 0; level < k; ++level) {
        int ones = (u % 3 == 1) + (v % 3 == 1) + (w % 3 == 1);
        if (ones >= 2) return 0;
        u /= 3; v /= 3; w /= 3;
    }
    return 1;
}

void orc_init_menger(orc_t *o, int k)
{
    const int L = o->L;
    int size = 1;
    for (int i = 0; i < k; ++i) size *= 3;
    const int nT = (L + size - 1) / size;
    uint32_t key[2] = { (uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32) };
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                uint64_t T = ((uint64_t)(z / size) * (uint64_t)nT + (uint64_t)(y / size)) * (uint64_t)nT
                           + (uint64_t)(x / size);
                uint32_t ctr[4] = { (uint32_t)(T >> 7), (uint32_t)k, 0u, 3u };
                uint32_t out[4];
                orc_philox4x32_10(ctr, key, out);
                int bit = (int)((out[(T >> 5) & 3] >> (T & 31)) & 1u);
                int sign = bit ? 1 : -1;
                int solid = orc_menger_solid(x % size, y % size, z % size, k);
                o->s[orc_idx(o, x, y, z)] = (int8_t)(solid ? sign : -sign);
            }
    o->sweep = 0;
}

/* The same start for one site (D11 written out for (x,y,z) alone): for */
/* sampled-site parity at sizes where the array version is too slow     */
/* (L = 2048, k = 0: the tile index passes 2^32).  Pinned against       */
/* orc_init_menger site by site on small L and against the big-integer  */
/* Python Philox on hand-indexed tiles of L = 2048 (test_oracle_next).  */
int orc_menger_site(uint64_t seed, int L, int k, int x, int y, int z)
{
    int size = 1;
    for (int i = 0; i < k; ++i) size *= 3;
    const uint64_t nT = (uint64_t)((L + size - 1) / size);
    const uint64_t T = ((uint64_t)(z / size) * nT + (uint64_t)(y / size)) * nT + (uint64_t)(x / size);
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)(T >> 7), (uint32_t)k, 0u, 3u };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    const int sign = ((out[(T >> 5) & 3] >> (T & 31)) & 1u) ? 1 : -1;
    return orc_menger_solid(x % size, y % size, z % size, k) ? sign : -sign;
}

/* ------------------------------------------------------------------ */
/* Finite-temperature Glauber dynamics (eq. (5)       */
/* PAPER.md:101): a proposed flip is accepted with probability          */
/*     p_acc(Delta E, T) = 1 / (1 + exp(Delta E / T)),   k_B = 1,        */
/* Delta E = 2 s_i sum_nn s_j = 12 - 4n (n antiparallel neighbours).     */
/* Reading D13 (the paper does not run T > 0 and names no RNG): each     */
/* site draws a 32-bit uniform u per sweep, u = sum_j b_j 2^(31-j) with  */
/* b_j the site's bit of Philox(key = seed, counter = (q, t, c, 4 + j)), */
/* j = 0..31 (one Philox call yields bit j of u for the 128 spins of a   */
/* group); the flip is accepted iff u < thr[n], thr[n] =                 */
/* floor(p_acc(12 - 4n, T) * 2^32) as a 64-bit integer in [0, 2^32]      */
/* (p = 1 always accepts), computed in fp64 with the C library's exp().  */
/* Sweep order as at T = 0 (colour 0, then colour 1).                    */
/* ------------------------------------------------------------------ */
void orc_glauber_thresholds(double T, uint64_t thr[7])
{
    for (int n = 0; n <= 6; ++n) {
        double dE = 12.0 - 4.0 * (double)n;
        double p = 1.0 / (1.0 + exp(dE / T));
        thr[n] = (uint64_t)floor(p * 4294967296.0);
    }
}

uint32_t orc_site_uniform(uint64_t seed, int L, int x, int y, int z, uint32_t t)
{
    uint32_t u = 0;
    for (uint32_t j = 0; j < 32; ++j)
        u |= (uint32_t)orc_site_bit(seed, L, x, y, z, t, 4u + j) << (31u - j);
    return u;
}

static inline void orc_update_site_T(orc_t *o, int x, int y, int z, uint32_t t, const uint64_t thr[7])
{
    const int L = o->L;
    int8_t *si = &o->s[orc_idx(o, x, y, z)];
    int n = 0;                                   /* antiparallel neighbours */
    n += o->s[orc_idx(o, orc_mod(x + 1, L), y, z)] != *si;
    n += o->s[orc_idx(o, orc_mod(x - 1, L), y, z)] != *si;
    n += o->s[orc_idx(o, x, orc_mod(y + 1, L), z)] != *si;
    n += o->s[orc_idx(o, x, orc_mod(y - 1, L), z)] != *si;
    n += o->s[orc_idx(o, x, y, orc_mod(z + 1, L))] != *si;
    n += o->s[orc_idx(o, x, y, orc_mod(z - 1, L))] != *si;
    if ((uint64_t)orc_site_uniform(o->seed, L, x, y, z, t) < thr[n]) *si = (int8_t)(-*si);
}

void orc_half_sweep_T(orc_t *o, uint32_t t, int c, const uint64_t thr[7])
{
    const int L = o->L;
    #pragma omp parallel for schedule(static)
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x)
                if (((x + y + z) & 1) == c) orc_update_site_T(o, x, y, z, t, thr);
}

void orc_sweep_T(orc_t *o, uint64_t n_sweeps, double T)
{
    uint64_t thr[7];
    orc_glauber_thresholds(T, thr);
    for (uint64_t i = 0; i < n_sweeps; ++i) {
        orc_half_sweep_T(o, o->sweep, 0, thr);
        orc_half_sweep_T(o, o->sweep, 1, thr);
        o->sweep += 1;
    }
}

/* ------------------------------------------------------------------ */
/* The paper's own estimator:      */
/* "C(r,t) shown in the main text is then obtained by radially          */
/* averaging over the three-dimensional correlation matrix" with the    */
/* matrix  [F^-1(|F s|^2)]_k = N * mean_i s_i s_{i+k}  (eq. 7).          */
/* Here the matrix is written from its definition, as the INTEGER       */
/*     P(d) = sum_i s_i s_{i+d},   d in [0,L)^3, periodic,               */
/* by direct double loops (O(N^2): tiny L only; for larger L the Python  */
/* wrapper takes the FFT route of eq. (7) in fp64 and rounds to the      */
/* integer, pinned against this function).                               */
/* Reading D12 (the paper does not define the radial average): the       */
/* displacement d is folded to the minimal image, each component in      */
/* (-L/2, L/2]; its bin is the integer b nearest to |d|, decided in      */
/* integers: (2b-1)^2 <= 4|d|^2 < (2b+1)^2; bins b = 0..L/2 are kept     */
/* (complete shells).  C_rad(b) = sum_{d in bin b} P(d) / (N * n(b))     */
/* - m^2, n(b) = number of displacements in the bin.                     */
/* ------------------------------------------------------------------ */
int orc_radial_bin(int L, int dx, int dy, int dz)
{
    /* fold to the minimal image, components in (-L/2, L/2] */
    if (dx > L / 2) dx -= L;
    if (dy > L / 2) dy -= L;
    if (dz > L / 2) dz -= L;
    int64_t n4 = 4 * ((int64_t)dx * dx + (int64_t)dy * dy + (int64_t)dz * dz);
    int64_t b = 0;
    while ((2 * b + 1) * (2 * b + 1) <= n4) ++b;       /* first b with 4|d|^2 < (2b+1)^2 */
    return (int)b;
}

/* P(d) for every d, direct definition.  out[(dz*L + dy)*L + dx], int64. */
void orc_corr_direct(const orc_t *o, int64_t *out)
{
    const int L = o->L;
    #pragma omp parallel for schedule(static)
    for (int dz = 0; dz < L; ++dz)
        for (int dy = 0; dy < L; ++dy)
            for (int dx = 0; dx < L; ++dx) {
                int64_t acc = 0;
                for (int z = 0; z < L; ++z)
                    for (int y = 0; y < L; ++y)
                        for (int x = 0; x < L; ++x)
                            acc += (int64_t)o->s[orc_idx(o, x, y, z)] *
                                   (int64_t)o->s[orc_idx(o, orc_mod(x + dx, L), orc_mod(y + dy, L),
                                                         orc_mod(z + dz, L))];
                out[((size_t)dz * L + dy) * L + dx] = acc;
            }
}

/* Radial sums of an integer field f[(dz*L + dy)*L + dx] over the bins of D12:
 * sum[b] = sum of f over bin b, cnt[b] = n(b), b = 0..L/2. */
void orc_radial_sums(int L, const int64_t *f, int64_t *sum, uint64_t *cnt)
{
    for (int b = 0; b <= L / 2; ++b) { sum[b] = 0; cnt[b] = 0; }
    for (int dz = 0; dz < L; ++dz)
        for (int dy = 0; dy < L; ++dy)
            for (int dx = 0; dx < L; ++dx) {
                int b = orc_radial_bin(L, dx, dy, dz);
                if (b <= L / 2) {
                    sum[b] += f[((size_t)dz * L + dy) * L + dx];
                    cnt[b] += 1;
                }
            }
}

/* ------------------------------------------------------------------ */
/* Brute-force variant for tiny L (pin P7): Delta E is obtained as     */
/* H(flipped configuration) - H(configuration), H = -sum over all 3N   */
/* bonds of s_i s_j (each bond once: +x, +y, +z neighbour of each site).*/
/* ------------------------------------------------------------------ */
int64_t orc_energy(const orc_t *o)
{
    const int L = o->L;
    int64_t H = 0;
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int s = o->s[orc_idx(o, x, y, z)];
                H -= s * o->s[orc_idx(o, orc_mod(x + 1, L), y, z)];
                H -= s * o->s[orc_idx(o, x, orc_mod(y + 1, L), z)];
                H -= s * o->s[orc_idx(o, x, y, orc_mod(z + 1, L))];
            }
    return H;
}

void orc_half_sweep_brute(orc_t *o, uint32_t t, int c)
{
    const int L = o->L;
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                if (((x + y + z) & 1) != c) continue;
                int8_t *si = &o->s[orc_idx(o, x, y, z)];
                int64_t H0 = orc_energy(o);
                *si = (int8_t)(-*si);
                int64_t H1 = orc_energy(o);
                int64_t dE = H1 - H0;
                int accept;
                if (dE < 0) accept = 1;
                else if (dE > 0) accept = 0;
                else accept = orc_site_bit(o->seed, L, x, y, z, t, 0u);
                if (!accept) *si = (int8_t)(-*si);
            }
}

void orc_sweep_brute(orc_t *o, uint64_t n_sweeps)
{
    for (uint64_t i = 0; i < n_sweeps; ++i) {
        orc_half_sweep_brute(o, o->sweep, 0);
        orc_half_sweep_brute(o, o->sweep, 1);
        o->sweep += 1;
    }
}

/* ------------------------------------------------------------------ */
/* D8 integer measurements.                                            */
/*   N_up = #{s = +1};                                                 */
/*   A_mu(r) = #{sites i : s_i != s_{i + r e_mu}}, mu = x,y,z, over    */
/*   ALL N sites i, periodic (eq. (2) PAPER.md:43 reduced to counts:   */
/*   s_i s_j = +1 / -1 for parallel / antiparallel pairs).             */
/* r_list[n_r] are the displacements wanted (0 <= r <= L/2);           */
/* antipar is [3][n_r], row-major, same order as r_list.               */
/* ------------------------------------------------------------------ */
void orc_measure(const orc_t *o, const int32_t *r_list, int n_r,
                 uint64_t *n_up, uint64_t *antipar)
{
    const int L = o->L;
    uint64_t up = 0;
    #pragma omp parallel for schedule(static) reduction(+:up)
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x)
                if (o->s[orc_idx(o, x, y, z)] == 1) up += 1;
    *n_up = up;

    for (int ir = 0; ir < n_r; ++ir) {
        const int r = r_list[ir];
        uint64_t ax = 0, ay = 0, az = 0;
        #pragma omp parallel for schedule(static) reduction(+:ax,ay,az)
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    int8_t s = o->s[orc_idx(o, x, y, z)];
                    if (s != o->s[orc_idx(o, orc_mod(x + r, L), y, z)]) ax += 1;
                    if (s != o->s[orc_idx(o, x, orc_mod(y + r, L), z)]) ay += 1;
                    if (s != o->s[orc_idx(o, x, y, orc_mod(z + r, L))]) az += 1;
                }
        antipar[0 * (size_t)n_r + ir] = ax;
        antipar[1 * (size_t)n_r + ir] = ay;
        antipar[2 * (size_t)n_r + ir] = az;
    }
}

/* ------------------------------------------------------------------ */
/* D9 fp64 post-processing of the counts, in exactly this order:       */
/*   m = (double)(2 N_up - N) / (double)N;                             */
/*   S(r) = 3N - 2 (A_x + A_y + A_z)(r)           (int64);             */
/*   C(r) = (double)S(r) / (double)(3N) - m*m     (eq. 2; */
/*          lattice average of one configuration, axis-averaged);      */
/*   ell: r0 = smallest r in [0, L/2-1] with C(r0) >= c > C(r0+1);     */
/*        ell = r0 + (C(r0) - c) / (C(r0) - C(r0+1))  (PAPER.md:51,    */
/*        linear interpolation); NaN if there is no such r0.           */
/* antipar is [3][L/2+1] here (all displacements).                     */
/* ------------------------------------------------------------------ */
void orc_postprocess(int L, uint64_t n_up, const uint64_t *antipar, double c_intercept,
                     double *m_out, double *C, double *ell)
{
    const int nr = L / 2 + 1;
    const int64_t N = (int64_t)L * L * L;
    double m = (double)(2 * (int64_t)n_up - N) / (double)N;
    *m_out = m;
    for (int r = 0; r < nr; ++r) {
        int64_t A = (int64_t)antipar[0 * nr + r] + (int64_t)antipar[1 * nr + r]
                  + (int64_t)antipar[2 * nr + r];
        int64_t S = 3 * N - 2 * A;
        C[r] = (double)S / (double)(3 * N) - m * m;
    }
    *ell = NAN;
    for (int r = 0; r + 1 < nr; ++r) {
        if (C[r] >= c_intercept && C[r + 1] < c_intercept) {
            *ell = (double)r + (C[r] - c_intercept) / (C[r] - C[r + 1]);
            break;
        }
    }
}

/* ------------------------------------------------------------------ */
/* D3 export / import: colour 0 words then colour 1 words; 32-bit      */
/* words, bit j (LSB = 0) of word w holds bit index b = 32 w + j;      */
/* bit value 1 <=> s = +1.                                             */
/* words per colour = ceil(L^3/2 / 32).                                */
/* ------------------------------------------------------------------ */
size_t orc_words_per_colour(int L)
{
    uint64_t bits = (uint64_t)L * L * L / 2;
    return (size_t)((bits + 31) / 32);
}

void orc_export(const orc_t *o, uint32_t *words)
{
    const int L = o->L;
    size_t wpc = orc_words_per_colour(L);
    memset(words, 0, 2 * wpc * sizeof(uint32_t));
    /* rows of L/2 bits start on word boundaries when L % 64 == 0: planes then touch disjoint
     * words and may go in parallel (no arithmetic here, only the D3 format) */
    #pragma omp parallel for schedule(static) if (L % 64 == 0)
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int c = (x + y + z) & 1;
                uint64_t b = orc_bit_index(L, x, y, z);
                if (o->s[orc_idx(o, x, y, z)] == 1)
                    words[(size_t)c * wpc + (size_t)(b >> 5)] |= (1u << (b & 31));
            }
}

void orc_import(orc_t *o, const uint32_t *words, uint32_t sweep)
{
    const int L = o->L;
    size_t wpc = orc_words_per_colour(L);
    #pragma omp parallel for schedule(static)
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int c = (x + y + z) & 1;
                uint64_t b = orc_bit_index(L, x, y, z);
                uint32_t bit = (words[(size_t)c * wpc + (size_t)(b >> 5)] >> (b & 31)) & 1u;
                o->s[orc_idx(o, x, y, z)] = bit ? (int8_t)1 : (int8_t)-1;
            }
    o->sweep = sweep;
}

/* ------------------------------------------------------------------ */
/* One site, computed one by one from the definition alone (no lattice */
/* array): the value of site (x,y,z) after h half-sweeps from the      */
/* T = infinity start of `seed`, by recursion over its light cone.     */
/* Half-sweep number i = 1,2,... belongs to sweep t = (i-1)/2 and      */
/* updates colour (i-1) mod 2 (D7).  Cost 7^h Philox calls: meant for  */
/* sampled sites of lattices too large for the array version (L=2048). */
/* Pinned against orc_sweep on small L (tests/test_oracle_pins.py).    */
/* ------------------------------------------------------------------ */
int orc_site_after(uint64_t seed, int L, int x, int y, int z, int h)
{
    if (h == 0) return orc_site_bit(seed, L, x, y, z, 0u, 1u) ? 1 : -1;
    const int c = (x + y + z) & 1;
    const int colour_updated = (h - 1) & 1;
    const uint32_t t = (uint32_t)((h - 1) / 2);
    const int s = orc_site_after(seed, L, x, y, z, h - 1);
    if (colour_updated != c) return s;
    const int sum = orc_site_after(seed, L, orc_mod(x + 1, L), y, z, h - 1)
                  + orc_site_after(seed, L, orc_mod(x - 1, L), y, z, h - 1)
                  + orc_site_after(seed, L, x, orc_mod(y + 1, L), z, h - 1)
                  + orc_site_after(seed, L, x, orc_mod(y - 1, L), z, h - 1)
                  + orc_site_after(seed, L, x, y, orc_mod(z + 1, L), h - 1)
                  + orc_site_after(seed, L, x, y, orc_mod(z - 1, L), h - 1);
    const int dE = 2 * s * sum;
    if (dE < 0) return -s;
    if (dE > 0) return s;
    return orc_site_bit(seed, L, x, y, z, t, 0u) ? -s : s;
}

/* same for a list of sites, in parallel over the list */
void orc_sites_after(uint64_t seed, int L, const int32_t *xyz, int n, int h, int8_t *out)
{
    #pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < n; ++i)
        out[i] = (int8_t)orc_site_after(seed, L, xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], h);
}

/* how many threads the OpenMP loops above use (bench.py reports it) */
#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
void orc_set_num_threads(int n) { omp_set_num_threads(n); }
#else
int orc_num_threads(void) { return 1; }
void orc_set_num_threads(int n) { (void)n; }
#endif
