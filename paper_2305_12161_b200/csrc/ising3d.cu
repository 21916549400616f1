// libising3d: C ABI (include/ising3d.h) + host launch layer.
// No CPU fallback anywhere: every compute entry point launches CUDA kernels or fails.
#include "../../include/ising3d.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>
#include <cufft.h>

#include "kernels_fused.cuh"
#include "kernels_fused2.cuh"
#include "kernels_fused3.cuh"
#include "kernels_active.cuh"
#include "kernels_generic.cuh"
#include "kernels_fft.cuh"
#include "kernels_gram.cuh"
#include "kernels_measure.cuh"
#include "kernels_resident.cuh"
#include "philox.cuh"

namespace {

thread_local std::string g_last_error = "";

int fail(int code, const std::string &msg)
{
    g_last_error = msg;
    return code;
}

#define CUDA_TRY(expr)                                                                     \
    do {                                                                                   \
        cudaError_t err__ = (expr);                                                        \
        if (err__ != cudaSuccess)                                                          \
            return fail(err__ == cudaErrorMemoryAllocation ? ISING3D_ENOMEM : ISING3D_ECUDA, \
                        std::string(#expr) + ": " + cudaGetErrorString(err__));            \
    } while (0)

bool valid_shape(int L, int n_rep) { return L >= 64 && L <= 4096 && (L % 64) == 0 && n_rep >= 1; }

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

constexpr int kActStride = 8;    // 64-bit counters per replica in d_act

struct ising3d {
    int L = 0, n_rep = 0;
    uint64_t sweep = 0;
    std::vector<uint64_t> seeds;
    cudaStream_t stream = nullptr;
    bool owns_mem = false;
    void *base = nullptr;
    uint32_t *state[2] = {nullptr, nullptr};   // ping-pong buffers (the fused kernel writes the other one)
    int cur = 0;
    uint64_t *d_seeds = nullptr;
    unsigned long long *d_counts = nullptr;
    int variant = ISING3D_VARIANT_AUTO;
    int cycle = ISING3D_CYCLE_01;
    int measure_variant = ISING3D_MEASURE_AUTO;
    double temperature = 0.0;                  // 0 = the paper's T -> 0 rule (eq. 6); > 0: eq. (5), D13
    ising::GlauberTables glauber = {};
    unsigned long long *d_gsum = nullptr;      // [n_rep][3][L/2+1] Gram diagonal sums
    unsigned int *d_queue = nullptr;           // [3 n_rep] task counters of gram_kernel
    // FFT estimator (ising3d_measure_radial): created on first use, library-owned
    double *fft_buf = nullptr;                 // [L][L][L+2] in-place real / half-complex field
    void *fft_work = nullptr;                  // cuFFT work area shared by both plans
    unsigned long long *d_rad = nullptr;       // [2][L/2+1] P sums, shell counts; [L/2+1] doubles; max rounding distance
    double radial_rounding = -1.0;             // max |v/N - llrint(v/N)| of the last measure_radial call
    cufftHandle plan_fwd = 0, plan_inv = 0;
    bool fft_ready = false;
    uint64_t launches = 0;
    int sm_count = 148;
    mutable ising::ResidentPlan res_plan = {0, 0};
    mutable bool res_planned = false;
    // launch shapes and per-device function attributes, set up at the handle's first use of a
    // kernel (nothing process-wide: distinct handles are independent, include/ising3d.h)
    ising::FusedPlan plan_f1, plan_f2, plan_f3;
    bool attr_gram = false, attr_autocorr = false;
    // activity-driven sweeps (kernels_active.cuh): one flag per 128-spin group and colour
    uint32_t *d_awake = nullptr;               // [n_rep][2][G/32]; valid only while flags_valid
    unsigned long long *d_act = nullptr;       // [n_rep][kActStride]: flag counts of colour 0, 1; groups evaluated,
                                               // changed; groups found holding a Delta E <= 0 site (probe tally)
    unsigned int *d_tickets = nullptr;         // work-item counter of active_halfsweep_kernel (never reset)
    uint32_t *d_ff = nullptr;                  // [n_rep][(L/8)^3/32] block-order bits of the current sweep (D15, fused2)
    ising::ActivePlan plan_act;
    bool flags_valid = false;                  // the flags describe state[cur] (set by activity_flags, kept by active sweeps)
    bool active_mode = false;                  // AUTO: the activity-driven kernel is the one being dispatched
    uint64_t run_len = 0;                      // sweeps since the last probe / check (AUTO)
    uint64_t probe_interval = 1024;            // AUTO: dense sweeps between two activity probes (0 = never)
    double active_on = 0.11, active_off = 0.14;   // AUTO: switch on below / off above this awake fraction
    double last_activity = -1.0;               // awake fraction seen by the last probe / check
    // AUTO probes never block the host: counts are copied to pinned memory, an event marks the copy,
    // and the enqueue loop looks at the event (cudaEventQuery) between launches
    unsigned long long *h_probe = nullptr;     // pinned, [n_rep][kActStride]
    cudaEvent_t probe_event = nullptr;
    bool probe_pending = false;                // a probe is in flight on the stream
    bool probe_stale = false;                  // ... but the state was replaced since: drop its result
    bool probe_active = false;                 // it was taken in active mode (tally) / dense mode (flag counts)
    uint64_t probe_sweeps = 0;                 // sweeps the active-mode tally of that probe covers
    uint64_t tally_sweeps = 0;                 // active-mode sweeps enqueued since the tally was last cleared

    size_t words_per_replica() const { return (size_t)L * L * L / 32; }
    size_t state_bytes() const { return words_per_replica() * 4 * (size_t)n_rep; }
    int counts_per_replica() const { return 1 + 3 * (L / 2 + 1); }
    bool fused_ok() const { return ising::fused_supported(L); }
    bool fused2_ok() const { return ising::fused2_supported(L); }
    bool use_gram() const
    {
        return measure_variant == ISING3D_MEASURE_TENSOR ||
               (measure_variant == ISING3D_MEASURE_AUTO && ising::gram_supported(L));
    }
    bool resident_ok() const
    {
        if (!ising::resident_supported(L)) return false;
        if (!res_planned) {
            res_plan = ising::resident_plan(L, n_rep, sm_count);
            res_planned = true;
        }
        return res_plan.cs > 0;
    }
    bool use_resident() const
    {
        if (cycle == ISING3D_CYCLE_DOUBLE_CB_MIXED) return false;   // generic kernel only
        return variant == ISING3D_VARIANT_RESIDENT ||
               (variant == ISING3D_VARIANT_AUTO && resident_ok());
    }
    bool fused3_ok() const { return ising::fused3_supported(L); }
    bool use_fused3() const { return variant == ISING3D_VARIANT_FUSED3 && cycle == ISING3D_CYCLE_01; }
    bool use_fused2() const
    {
        return variant == ISING3D_VARIANT_FUSED2 || variant == ISING3D_VARIANT_FUSED3 ||
               (variant == ISING3D_VARIANT_AUTO && fused2_ok());
    }
    bool active_ok() const { return ising::active_supported(L); }
    bool use_active() const      // forced; AUTO switches to it by itself (sweep_auto)
    {
        return variant == ISING3D_VARIANT_ACTIVE && cycle <= ISING3D_CYCLE_MIXED && temperature == 0.0;
    }
    bool auto_adaptive() const
    {
        return variant == ISING3D_VARIANT_AUTO && fused2_ok() && active_ok() && cycle <= ISING3D_CYCLE_MIXED &&
               temperature == 0.0 && probe_interval > 0;
    }
    void state_changed()         // the state was replaced: flags and the adaptive history are void
    {
        flags_valid = false;
        active_mode = false;
        run_len = 0;
        last_activity = -1.0;
        probe_stale = probe_pending;
    }
    size_t flag_words() const { return (size_t)L * L * (L >> 8) / 32; }   // per colour
    bool use_fused() const
    {
        if (cycle != ISING3D_CYCLE_01) return false;
        return variant == ISING3D_VARIANT_FUSED ||
               (variant == ISING3D_VARIANT_AUTO && fused_ok() && !fused2_ok() && !resident_ok());
    }
};

namespace {

struct Layout {
    size_t state, seeds, counts, gsum, queue, awake, act, ff, total;
};

Layout make_layout(int L, int n_rep)
{
    Layout l;
    l.state = align_up((size_t)L * L * L / 8 * (size_t)n_rep, 256);
    l.seeds = align_up((size_t)n_rep * 8, 256);
    l.counts = align_up((size_t)n_rep * (1 + 3 * (L / 2 + 1)) * 8, 256);
    l.gsum = align_up((size_t)n_rep * 3 * (L / 2 + 1) * 8, 256);
    l.queue = align_up((size_t)n_rep * 3 * 4, 256);
    const bool act = ising::active_supported(L);
    l.awake = act ? align_up((size_t)n_rep * 2 * ((size_t)L * L * (L >> 8) / 8), 256) : 0;
    l.act = act ? align_up((size_t)n_rep * kActStride * 8, 256) + 256 : 0;        // + the ticket counter
    l.ff = ising::fused2_supported(L) ? align_up((size_t)n_rep * ((size_t)(L / 8) * (L / 8) * (L / 8) / 8), 256) : 0;
    l.total = 2 * l.state + l.seeds + l.counts + l.gsum + l.queue + l.awake + l.act + l.ff;
    return l;
}

int launch_init(ising3d *h)
{
    const size_t groups = h->words_per_replica() / 4;
    dim3 grid((unsigned)((groups + 255) / 256), (unsigned)h->n_rep);
    ising::init_spins_kernel<<<grid, 256, 0, h->stream>>>(h->state[h->cur], h->d_seeds, h->L);
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    h->sweep = 0;
    h->state_changed();
    return ISING3D_OK;
}

int create(ising3d_t **out, int L, int n_rep, const uint64_t *seeds, void *dev_buf,
           size_t dev_bytes, void *stream)
{
    if (!out || !seeds) return fail(ISING3D_EINVAL, "null pointer");
    if (!valid_shape(L, n_rep))
        return fail(ISING3D_EINVAL, "L must be a multiple of 64 in [64, 4096] and n_rep >= 1");
    if ((size_t)n_rep > 65535) return fail(ISING3D_EINVAL, "n_rep must be <= 65535");
    const Layout lay = make_layout(L, n_rep);
    ising3d *h = new (std::nothrow) ising3d();
    if (!h) return fail(ISING3D_ENOMEM, "host allocation failed");
    h->L = L;
    h->n_rep = n_rep;
    h->seeds.assign(seeds, seeds + n_rep);
    h->stream = (cudaStream_t)stream;
    int code = ISING3D_OK;
    do {
        cudaError_t e;
        if (dev_buf) {
            if (dev_bytes < lay.total || ((uintptr_t)dev_buf & 255)) {
                code = fail(ISING3D_EINVAL, "device buffer too small or not 256-byte aligned");
                break;
            }
            h->base = dev_buf;
            h->owns_mem = false;
        } else {
            e = cudaMalloc(&h->base, lay.total);
            if (e != cudaSuccess) {
                code = fail(e == cudaErrorMemoryAllocation ? ISING3D_ENOMEM : ISING3D_ECUDA,
                            std::string("cudaMalloc: ") + cudaGetErrorString(e));
                cudaGetLastError();
                break;
            }
            h->owns_mem = true;
        }
        char *p = (char *)h->base;
        h->state[0] = (uint32_t *)p;
        h->state[1] = (uint32_t *)(p + lay.state);
        h->d_seeds = (uint64_t *)(p + 2 * lay.state);
        h->d_counts = (unsigned long long *)(p + 2 * lay.state + lay.seeds);
        h->d_gsum = (unsigned long long *)(p + 2 * lay.state + lay.seeds + lay.counts);
        h->d_queue = (unsigned int *)(p + 2 * lay.state + lay.seeds + lay.counts + lay.gsum);
        if (lay.awake) {
            h->d_awake = (uint32_t *)(p + 2 * lay.state + lay.seeds + lay.counts + lay.gsum + lay.queue);
            h->d_act = (unsigned long long *)(p + 2 * lay.state + lay.seeds + lay.counts + lay.gsum +
                                              lay.queue + lay.awake);
            h->d_tickets = (unsigned int *)((char *)h->d_act + lay.act - 256);
        }
        if (lay.ff)
            h->d_ff = (uint32_t *)(p + 2 * lay.state + lay.seeds + lay.counts + lay.gsum + lay.queue + lay.awake +
                                   lay.act);
        int dev = 0;
        if ((e = cudaGetDevice(&dev)) != cudaSuccess ||
            (e = cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev)) !=
                cudaSuccess ||
            (e = cudaMemcpyAsync(h->d_seeds, h->seeds.data(), (size_t)n_rep * 8,
                                 cudaMemcpyHostToDevice, h->stream)) != cudaSuccess) {
            code = fail(ISING3D_ECUDA, std::string("setup: ") + cudaGetErrorString(e));
            break;
        }
        if (h->d_act && (e = cudaMemsetAsync(h->d_act, 0, lay.act, h->stream)) != cudaSuccess) {
            code = fail(ISING3D_ECUDA, std::string("setup: ") + cudaGetErrorString(e));
            break;
        }
        if (h->d_act && lay.ff &&
            ((e = cudaHostAlloc((void **)&h->h_probe, (size_t)n_rep * kActStride * 8, cudaHostAllocDefault)) != cudaSuccess ||
             (e = cudaEventCreateWithFlags(&h->probe_event, cudaEventDisableTiming)) != cudaSuccess)) {
            code = fail(ISING3D_ECUDA, std::string("setup (probe buffer): ") + cudaGetErrorString(e));
            break;
        }
        // the seeds vector outlives the copy (it lives in the handle)
        code = launch_init(h);
    } while (0);
    if (code != ISING3D_OK) {
        if (h->owns_mem && h->base) cudaFree(h->base);
        if (h->h_probe) cudaFreeHost(h->h_probe);
        if (h->probe_event) cudaEventDestroy(h->probe_event);
        cudaGetLastError();
        delete h;
        return code;
    }
    *out = h;
    return ISING3D_OK;
}

int sweep_generic(ising3d *h, uint64_t n)
{
    const size_t groups = h->words_per_replica() / 8;   // per colour
    dim3 grid((unsigned)((groups + 255) / 256), (unsigned)h->n_rep);
    const int mixed = h->cycle == ISING3D_CYCLE_MIXED;
    for (uint64_t i = 0; i < n; ++i) {
        const uint32_t t = (uint32_t)(h->sweep + i);
        if (h->cycle == ISING3D_CYCLE_DOUBLE_CB_MIXED) {
            // D15: draw the blocks' fine orders into the idle ping-pong buffer, then for the two
            // coarse colours in the drawn order: pass 0 (each block's first fine colour), pass 1
            uint32_t *ff = h->state[1 - h->cur];
            const size_t stride = h->words_per_replica();
            const int nB = h->L / 8, n_words = nB * nB * nB / 32;
            ising::block_order_kernel<<<dim3((unsigned)((n_words + 255) / 256), (unsigned)h->n_rep), 256, 0,
                                        h->stream>>>(ff, stride, h->d_seeds, n_words, t);
            for (int k = 0; k < 2; ++k)
                for (int pass = 0; pass < 2; ++pass)
                    for (int c = 0; c < 2; ++c)
                        ising::halfsweep_generic_kernel<<<grid, 256, 0, h->stream>>>(
                            h->state[h->cur], h->d_seeds, h->L, t, c, 0, k, ff, stride, pass);
            h->launches += 7;
            continue;
        }
        if (h->cycle == ISING3D_CYCLE_DOUBLE_CB) {
            // red blocks: dark sites, light sites; then the blue blocks (Supp. I.A, D14)
            for (int coarse = 0; coarse < 2; ++coarse)
                for (int fine = 0; fine < 2; ++fine)
                    ising::halfsweep_generic_kernel<<<grid, 256, 0, h->stream>>>(
                        h->state[h->cur], h->d_seeds, h->L, t, fine, 0, coarse);
            h->launches += 2;
            continue;
        }
        ising::halfsweep_generic_kernel<<<grid, 256, 0, h->stream>>>(h->state[h->cur], h->d_seeds,
                                                                     h->L, t, 0, mixed, -1);
        ising::halfsweep_generic_kernel<<<grid, 256, 0, h->stream>>>(h->state[h->cur], h->d_seeds,
                                                                     h->L, t, 1, mixed, -1);
    }
    h->launches += 2 * n;
    CUDA_TRY(cudaGetLastError());
    return ISING3D_OK;
}

int sweep_glauber(ising3d *h, uint64_t n)
{
    const size_t groups = h->words_per_replica() / 8;   // per colour
    dim3 grid((unsigned)((groups + 255) / 256), (unsigned)h->n_rep);
    const int mixed = h->cycle == ISING3D_CYCLE_MIXED;
    for (uint64_t i = 0; i < n; ++i) {
        const uint32_t t = (uint32_t)(h->sweep + i);
        ising::halfsweep_glauber_kernel<<<grid, 256, 0, h->stream>>>(h->state[h->cur], h->d_seeds, h->L,
                                                                     t, 0, mixed, h->glauber);
        ising::halfsweep_glauber_kernel<<<grid, 256, 0, h->stream>>>(h->state[h->cur], h->d_seeds, h->L,
                                                                     t, 1, mixed, h->glauber);
    }
    h->launches += 2 * n;
    CUDA_TRY(cudaGetLastError());
    return ISING3D_OK;
}

int sweep_resident(ising3d *h, uint64_t n)
{
    cudaError_t e = ising::launch_resident(h->state[h->cur], h->d_seeds, h->L, h->n_rep, h->res_plan,
                                           (uint32_t)h->sweep, (uint32_t)n, h->cycle, h->stream);
    if (e != cudaSuccess)
        return fail(ISING3D_ECUDA, std::string("resident sweep launch: ") + cudaGetErrorString(e));
    h->launches += 1;
    return ISING3D_OK;
}

// One launch per replica and sweep (pair of sweeps for fused3): the replicas of a batch are
// independent lattices at a stride of words_per_replica() in both ping-pong buffers.
// Runs the sweeps with indices h->sweep + i0 .. h->sweep + i0 + n - 1.
int sweep_fused(ising3d *h, uint64_t i0, uint64_t n, bool gen2)
{
    const size_t wpr = h->words_per_replica();
    uint64_t i = 0;
    {
        cudaError_t e = cudaSuccess;
        if (gen2 && !h->plan_f2.ready) e = ising::plan_fused2(h->plan_f2, h->L, h->sm_count);
        if (e == cudaSuccess && !gen2 && !h->plan_f1.ready) e = ising::plan_fused(h->plan_f1, h->L, h->sm_count);
        if (e == cudaSuccess && gen2 && h->use_fused3() && !h->plan_f3.ready)
            e = ising::plan_fused3(h->plan_f3, h->L, h->sm_count);
        if (e != cudaSuccess)
            return fail(ISING3D_ECUDA, std::string("fused sweep plan: ") + cudaGetErrorString(e));
    }
    if (n) h->flags_valid = false;             // the dense kernels do not keep the activity flags
    // pairs of sweeps with the intermediate state on chip (01 cycle); an odd last sweep below
    for (; gen2 && h->use_fused3() && i + 2 <= n; i += 2) {
        for (int rep = 0; rep < h->n_rep; ++rep) {
            cudaError_t e = ising::launch_fused3_sweep2(
                h->state[h->cur] + rep * wpr, h->state[1 - h->cur] + rep * wpr, h->L,
                (uint32_t)(h->sweep + i0 + i), h->seeds[rep], h->plan_f3, h->stream);
            if (e != cudaSuccess)
                return fail(ISING3D_ECUDA, std::string("fused3 sweep launch: ") + cudaGetErrorString(e));
        }
        h->cur = 1 - h->cur;
        h->launches += h->n_rep;
    }
    const bool dcbm = gen2 && h->cycle == ISING3D_CYCLE_DOUBLE_CB_MIXED;
    const int nB = h->L / 8, ff_words = nB * nB * nB / 32;
    for (; i < n; ++i) {
        const uint32_t t = (uint32_t)(h->sweep + i0 + i);
        if (dcbm) {     // D15: this sweep's fine order of every block, all replicas
            ising::block_order_kernel<<<dim3((unsigned)((ff_words + 255) / 256), (unsigned)h->n_rep), 256, 0,
                                        h->stream>>>(h->d_ff, (size_t)ff_words, h->d_seeds, ff_words, t);
            h->launches += 1;
        }
        for (int rep = 0; rep < h->n_rep; ++rep) {
            const uint64_t seed = h->seeds[rep];
            const uint32_t *src = h->state[h->cur] + rep * wpr;
            uint32_t *dst = h->state[1 - h->cur] + rep * wpr;
            // mixed cycle (D10): the launch layer draws this sweep's first colour on the host
            const int first = h->cycle == ISING3D_CYCLE_MIXED ? ising::first_colour(seed, t) : 0;
            cudaError_t e;
            if (dcbm) {
                // D15: the coarse colours in the drawn order; for each, the blocks that drew "dark first"
                // and the blocks that drew "light first" in one masked launch each (blocks of one coarse
                // colour do not touch): src -> dst -> src -> dst -> src
                const uint32_t *ffr = h->d_ff + (size_t)rep * ff_words;
                uint32_t *a = const_cast<uint32_t *>(src), *b = dst;
                e = cudaSuccess;
                for (int k = 0; k < 2 && e == cudaSuccess; ++k)
                    for (int f = 0; f < 2 && e == cudaSuccess; ++f) {
                        e = ising::launch_fused2_sweep(a, b, h->L, t, seed, f, h->plan_f2, h->stream,
                                                       k ^ ising::first_colour(seed, t), ffr);
                        std::swap(a, b);
                    }
            } else if (gen2 && h->cycle == ISING3D_CYCLE_DOUBLE_CB) {
                // D14: the red blocks (dark, then light sites), then the blue blocks: two masked
                // launches, src -> dst -> src
                e = ising::launch_fused2_sweep(src, dst, h->L, t, seed, 0, h->plan_f2, h->stream, 0);
                if (e == cudaSuccess)
                    e = ising::launch_fused2_sweep(dst, const_cast<uint32_t *>(src), h->L, t, seed, 0,
                                                   h->plan_f2, h->stream, 1);
            } else {
                e = gen2 ? ising::launch_fused2_sweep(src, dst, h->L, t, seed, first, h->plan_f2, h->stream)
                         : ising::launch_fused_sweep(src, dst, h->L, t, ising::make_philox_keys(seed),
                                                     h->plan_f1, h->stream);
            }
            if (e != cudaSuccess)
                return fail(ISING3D_ECUDA, std::string("fused sweep launch: ") + cudaGetErrorString(e));
        }
        if (dcbm) {
            h->launches += 4 * (uint64_t)h->n_rep;         // back in state[cur]
        } else if (gen2 && h->cycle == ISING3D_CYCLE_DOUBLE_CB) {
            h->launches += 2 * (uint64_t)h->n_rep;         // back in state[cur]
        } else {
            h->cur = 1 - h->cur;
            h->launches += h->n_rep;
        }
    }
    CUDA_TRY(cudaGetLastError());
    return ISING3D_OK;
}

// Activity flags of state[cur] (kernels_active.cuh): flag = the group holds a site with Delta E <= 0
// (eq. (6)).  Counts land in d_act[rep][0..1].
int build_flags(ising3d *h)
{
    const size_t wpr = h->words_per_replica(), fw = h->flag_words();
    CUDA_TRY(cudaMemset2DAsync(h->d_act, kActStride * 8, 0, 2 * 8, (size_t)h->n_rep, h->stream));   // [rep][0..1]
    for (int rep = 0; rep < h->n_rep; ++rep) {
        cudaError_t e = ising::launch_activity_flags(h->state[h->cur] + rep * wpr, h->d_awake + rep * 2 * fw,
                                                     h->d_act + rep * kActStride, h->L, h->stream);
        if (e != cudaSuccess)
            return fail(ISING3D_ECUDA, std::string("activity flags launch: ") + cudaGetErrorString(e));
    }
    h->launches += h->n_rep;
    h->flags_valid = true;
    return ISING3D_OK;
}

// Synchronises the stream (ising3d_activity only; the AUTO probes go through probe_enqueue / probe_poll).
// frac = mean over replicas and colours of d_act[rep][0..1] / G;
// raw[rep][0..1] = the two counts.
int read_activity(ising3d *h, double *frac, uint64_t *raw)
{
    std::vector<unsigned long long> host((size_t)h->n_rep * kActStride);
    CUDA_TRY(cudaMemcpyAsync(host.data(), h->d_act, host.size() * 8, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    const double G = (double)h->flag_words() * 32.0;
    double sum = 0.0;
    for (int rep = 0; rep < h->n_rep; ++rep) {
        sum += (double)host[rep * kActStride + 0] + (double)host[rep * kActStride + 1];
        if (raw) {
            raw[rep * 2 + 0] = host[rep * kActStride + 0];
            raw[rep * 2 + 1] = host[rep * kActStride + 1];
        }
    }
    if (frac) *frac = sum / (2.0 * G * h->n_rep);
    return ISING3D_OK;
}

// Sweeps h->sweep + i0 .. + n - 1 on the activity-driven kernels, in place in state[cur].
int sweep_active(ising3d *h, uint64_t i0, uint64_t n)
{
    if (n == 0) return ISING3D_OK;
    if (!h->flags_valid) {
        const int rc = build_flags(h);
        if (rc != ISING3D_OK) return rc;
    }
    if (!h->plan_act.ready) {
        cudaError_t e = ising::plan_active(h->plan_act, h->L, h->sm_count);
        if (e != cudaSuccess) return fail(ISING3D_ECUDA, std::string("active sweep plan: ") + cudaGetErrorString(e));
    }
    const size_t wpr = h->words_per_replica(), fw = h->flag_words();
    for (uint64_t i = 0; i < n; ++i) {
        const uint32_t t = (uint32_t)(h->sweep + i0 + i);
        for (int rep = 0; rep < h->n_rep; ++rep) {
            const uint64_t seed = h->seeds[rep];
            const int first = h->cycle == ISING3D_CYCLE_MIXED ? ising::first_colour(seed, t) : 0;
            cudaError_t e = ising::launch_active_sweep(h->state[h->cur] + rep * wpr, h->d_awake + rep * 2 * fw,
                                                       h->d_act + rep * kActStride + 2, h->d_tickets, h->plan_act,
                                                       h->L, t, seed, first, h->stream);
            if (e != cudaSuccess) {
                // a refused launch leaves the host's ticket count and the flags in doubt: start both over
                ising::reset_active_tickets(h->d_tickets, h->plan_act, h->stream);
                h->flags_valid = false;
                return fail(ISING3D_ECUDA, std::string("active sweep launch: ") + cudaGetErrorString(e));
            }
        }
        h->launches += 2 * (uint64_t)h->n_rep;
    }
    return ISING3D_OK;
}

// ---- ISING3D_VARIANT_AUTO at L >= 512, T = 0, plain checkerboard -------------------------------------
// Dense fused2 sweeps while most groups still hold a site that can change, the activity-driven kernel
// once few do.  The choice changes the speed only, never the result, so it may lag: nothing here
// waits for the GPU.  Every probe_interval sweeps a probe is queued on the stream
//   dense mode:  rebuild the flags and count them (activity_flags_kernel), copy the counts to pinned memory
//   active mode: copy the kernel's own tally of groups found holding a Delta E <= 0 site, then clear it
// followed by an event; probe_poll looks at the event between launches and switches mode once a
// result has landed (on below active_on, off above active_off).  At most one probe is in flight.

// Clear the active-mode tally [rep][4] (stream ordered).
int clear_tally(ising3d *h)
{
    CUDA_TRY(cudaMemset2DAsync(h->d_act + 4, kActStride * 8, 0, 8, (size_t)h->n_rep, h->stream));
    h->tally_sweeps = 0;
    return ISING3D_OK;
}

int probe_poll(ising3d *h)
{
    if (!h->probe_pending) return ISING3D_OK;
    const cudaError_t q = cudaEventQuery(h->probe_event);
    if (q == cudaErrorNotReady) {
        cudaGetLastError();
        return ISING3D_OK;
    }
    h->probe_pending = false;
    if (q != cudaSuccess) return fail(ISING3D_ECUDA, std::string("activity probe: ") + cudaGetErrorString(q));
    if (h->probe_stale) {                       // taken on a state that has been replaced since
        h->probe_stale = false;
        return ISING3D_OK;
    }
    const double G = (double)h->flag_words() * 32.0;
    double sum = 0.0;
    for (int rep = 0; rep < h->n_rep; ++rep) {
        const unsigned long long *c = h->h_probe + (size_t)rep * kActStride;
        sum += h->probe_active ? (double)c[4] : (double)c[0] + (double)c[1];
    }
    // dense: flags set / all flags; active: groups that held such a site per colour update / groups per colour
    const double frac = sum / (2.0 * G * h->n_rep * (h->probe_active ? (double)h->probe_sweeps : 1.0));
    h->last_activity = frac;
    if (h->probe_active && h->active_mode && frac > h->active_off) {
        h->active_mode = false;
        h->run_len = 0;
    } else if (!h->probe_active && !h->active_mode && frac < h->active_on) {
        h->active_mode = true;
        h->run_len = 0;
        return clear_tally(h);                 // the tally counts from the first active sweep
    }
    return ISING3D_OK;
}

// Queue one probe after the sweeps enqueued so far.
int probe_enqueue(ising3d *h)
{
    if (h->probe_pending) return ISING3D_OK;   // the GPU has not reached the previous one yet
    if (h->active_mode && h->tally_sweeps == 0) return ISING3D_OK;
    const uint64_t sweeps = h->tally_sweeps;
    if (!h->active_mode) {
        const int rc = build_flags(h);
        if (rc != ISING3D_OK) return rc;
    }
    CUDA_TRY(cudaMemcpyAsync(h->h_probe, h->d_act, (size_t)h->n_rep * kActStride * 8, cudaMemcpyDeviceToHost,
                             h->stream));
    if (h->active_mode) {
        const int rc = clear_tally(h);
        if (rc != ISING3D_OK) return rc;
    }
    CUDA_TRY(cudaEventRecord(h->probe_event, h->stream));
    h->probe_pending = true;
    h->probe_stale = false;
    h->probe_active = h->active_mode;
    h->probe_sweeps = sweeps;
    return ISING3D_OK;
}

int sweep_auto(ising3d *h, uint64_t n)
{
    const uint64_t kPollEvery = 64;            // sweeps enqueued between two looks at the event
    // inside a stream capture: sweeps only, in the mode the handle is in (no event query, no probe)
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    CUDA_TRY(cudaStreamIsCapturing(h->stream, &cap));
    const bool probing = cap == cudaStreamCaptureStatusNone;
    uint64_t i = 0;
    while (i < n) {
        int rc = probing ? probe_poll(h) : ISING3D_OK;
        if (rc != ISING3D_OK) return rc;
        const uint64_t left = h->run_len < h->probe_interval ? h->probe_interval - h->run_len : 1;
        const uint64_t m = std::min<uint64_t>(std::min<uint64_t>(n - i, left), kPollEvery);
        rc = h->active_mode ? sweep_active(h, i, m) : sweep_fused(h, i, m, true);
        if (rc != ISING3D_OK) return rc;
        i += m;
        h->run_len += m;
        if (h->active_mode) h->tally_sweeps += m;
        if (h->run_len >= h->probe_interval) {
            rc = probing ? probe_enqueue(h) : ISING3D_OK;
            if (rc != ISING3D_OK) return rc;
            h->run_len = 0;
        }
    }
    return ISING3D_OK;
}

// D9: fp64 post-processing of the integer counts, in this exact order.
void postprocess(int L, uint64_t n_up, const uint64_t *antipar, double c_intercept, double *C,
                 double *ell)
{
    const int nr = L / 2 + 1;
    const int64_t N = (int64_t)L * L * L;
    const double m = (double)(2 * (int64_t)n_up - N) / (double)N;
    std::vector<double> tmp;
    if (!C) {
        tmp.resize(nr);
        C = tmp.data();
    }
    for (int r = 0; r < nr; ++r) {
        const int64_t A = (int64_t)antipar[r] + (int64_t)antipar[nr + r] + (int64_t)antipar[2 * nr + r];
        const int64_t S = 3 * N - 2 * A;
        C[r] = (double)S / (double)(3 * N) - m * m;
    }
    if (ell) {
        *ell = std::nan("");
        for (int r = 0; r + 1 < nr; ++r)
            if (C[r] >= c_intercept && C[r + 1] < c_intercept) {
                *ell = (double)r + (C[r] - c_intercept) / (C[r] - C[r + 1]);
                break;
            }
    }
}

// cuFFT plans and buffers of the radial estimator, on first use (8 bytes per site + work area)
int fft_setup(ising3d *h)
{
    if (h->fft_ready) return ISING3D_OK;
    const int L = h->L, H = L / 2 + 1;
    const size_t buf_bytes = (size_t)L * L * (L + 2) * sizeof(double);
    auto cleanup = [&]() {
        if (h->plan_fwd) cufftDestroy(h->plan_fwd);
        if (h->plan_inv) cufftDestroy(h->plan_inv);
        if (h->fft_buf) cudaFree(h->fft_buf);
        if (h->fft_work) cudaFree(h->fft_work);
        if (h->d_rad) cudaFree(h->d_rad);
        h->plan_fwd = h->plan_inv = 0;
        h->fft_buf = nullptr;
        h->fft_work = nullptr;
        h->d_rad = nullptr;
        cudaGetLastError();
    };
    size_t ws_f = 0, ws_i = 0;
    if (cudaMalloc(&h->fft_buf, buf_bytes) != cudaSuccess ||
        cudaMalloc(&h->d_rad, ((size_t)3 * H + 1) * 8) != cudaSuccess) {
        cleanup();
        return fail(ISING3D_ENOMEM, "radial estimator: cannot allocate the 8 bytes/site FFT field");
    }
    if (cufftCreate(&h->plan_fwd) != CUFFT_SUCCESS || cufftCreate(&h->plan_inv) != CUFFT_SUCCESS ||
        cufftSetAutoAllocation(h->plan_fwd, 0) != CUFFT_SUCCESS ||
        cufftSetAutoAllocation(h->plan_inv, 0) != CUFFT_SUCCESS ||
        cufftMakePlan3d(h->plan_fwd, L, L, L, CUFFT_D2Z, &ws_f) != CUFFT_SUCCESS ||
        cufftMakePlan3d(h->plan_inv, L, L, L, CUFFT_Z2D, &ws_i) != CUFFT_SUCCESS) {
        cleanup();
        return fail(ISING3D_ECUDA, "radial estimator: cuFFT plan creation failed");
    }
    const size_t ws = std::max(ws_f, ws_i);
    if (ws && cudaMalloc(&h->fft_work, ws) != cudaSuccess) {
        cleanup();
        return fail(ISING3D_ENOMEM, "radial estimator: cannot allocate the cuFFT work area");
    }
    if (cufftSetWorkArea(h->plan_fwd, h->fft_work) != CUFFT_SUCCESS ||
        cufftSetWorkArea(h->plan_inv, h->fft_work) != CUFFT_SUCCESS) {
        cleanup();
        return fail(ISING3D_ECUDA, "radial estimator: cufftSetWorkArea failed");
    }
    h->fft_ready = true;
    return ISING3D_OK;
}

// A_mu(r) on the tensor cores (kernels_gram.cuh): per replica and axis, gather the line words
// into the spare ping-pong buffer, run the Gram kernel, then A = 2 N_up - 2 Gsum.
int measure_gram(ising3d *h)
{
    const int L = h->L, nr = L / 2 + 1, cpr = h->counts_per_replica();
    const ising::GramPlan plan = ising::make_gram_plan(L, h->sm_count);
    const size_t smem = ising::gram_smem_bytes(L, plan);
    const int NWB = 4;                         // row words per block of the x gather
    const size_t smem_x = ((size_t)64 * NWB * (L / 32 + 1) + (size_t)2 * 256 * (NWB + 1)) * 4;
    if (!h->attr_gram) {       // per device, idempotent; once per handle
        CUDA_TRY(cudaFuncSetAttribute(ising::gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      210 * 1024));
        CUDA_TRY(cudaFuncSetAttribute(ising::gather_lines_x_kernel,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
        h->attr_gram = true;
    }
    CUDA_TRY(cudaMemsetAsync(h->d_gsum, 0, (size_t)h->n_rep * 3 * nr * 8, h->stream));
    CUDA_TRY(cudaMemsetAsync(h->d_queue, 0, (size_t)h->n_rep * 3 * 4, h->stream));
    const size_t wpr = h->words_per_replica();
    const int WPR = L >> 6;
    for (int rep = 0; rep < h->n_rep; ++rep) {
        const uint32_t *st = h->state[h->cur] + (size_t)rep * wpr;
        uint32_t *xw = h->state[1 - h->cur] + (size_t)rep * wpr;       // scratch: the other buffer
        for (int ax = 0; ax < 3; ++ax) {
            if (ax == 0)
                ising::gather_lines_x_kernel<<<(unsigned)(L * (WPR / NWB)), 256, smem_x, h->stream>>>(st, xw, L, NWB);
            else if (ax == 1)
                ising::gather_lines_yz_kernel<1><<<h->sm_count * 8, 256, 0, h->stream>>>(st, xw, L);
            else
                ising::gather_lines_yz_kernel<2><<<h->sm_count * 8, 256, 0, h->stream>>>(st, xw, L);
            ising::gram_kernel<<<h->sm_count, ising::kGramThreads, smem, h->stream>>>(
                xw, h->d_gsum + ((size_t)rep * 3 + ax) * nr, h->d_queue + rep * 3 + ax, L, plan);
            h->launches += 2;
        }
        ising::gram_finalize_kernel<<<(3 * nr + 255) / 256, 256, 0, h->stream>>>(
            h->d_counts + (size_t)rep * cpr, h->d_gsum + (size_t)rep * 3 * nr, nr);
        h->launches += 1;
    }
    CUDA_TRY(cudaGetLastError());
    return ISING3D_OK;
}

}  // namespace

// ---- ising3d_measure_static: the measurement with its accumulators in library-static memory --------
// The 64-bit counters count_up_kernel and autocorr_kernel add into ([rep][1 + 3 (L/2+1)], the layout at
// the top of kernels_measure.cuh).  Part of the loaded module: every GPU that loads the library holds
// these 128 KiB until the process exits; all calls on one GPU share them.
// In HOST code this name is only a stand-in for the device object, not a device address: it must never
// be handed to a kernel.  static_scratch_for_current_device() asks the runtime for the real address.
static __device__ __align__(256) unsigned long long g_static_counts[ISING3D_STATIC_MAX_COUNTS];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned long long *g_static_ptr[kStaticMaxDevices] = {};   // device address of g_static_counts, per device

// Once per device, with that device current: the device address of g_static_counts and the
// shared-memory opt-in of the three autocorr kernels (a per-device function attribute).  No allocation.
int static_scratch_for_current_device(unsigned long long **out)
{
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(ISING3D_EINVAL, "device ordinal out of range");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        unsigned long long *p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_static_counts));
        const int max_smem = (int)ising::autocorr_smem_bytes(4096, 8) + 4096;
        CUDA_TRY(cudaFuncSetAttribute(ising::autocorr_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
        CUDA_TRY(cudaFuncSetAttribute(ising::autocorr_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
        CUDA_TRY(cudaFuncSetAttribute(ising::autocorr_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return ISING3D_OK;
}

}  // namespace

extern "C" {

size_t ising3d_required_bytes(int L, int n_rep)
{
    if (!valid_shape(L, n_rep)) return 0;
    return make_layout(L, n_rep).total;
}

size_t ising3d_words_per_replica(int L)
{
    if (!valid_shape(L, 1)) return 0;
    return (size_t)L * L * L / 32;
}

int ising3d_init(ising3d_t **h, int L, uint64_t seed)
{
    return create(h, L, 1, &seed, nullptr, 0, nullptr);
}

int ising3d_init_batch(ising3d_t **h, int L, int n_rep, const uint64_t *seeds)
{
    return create(h, L, n_rep, seeds, nullptr, 0, nullptr);
}

int ising3d_init_batch_with_buffer(ising3d_t **h, int L, int n_rep, const uint64_t *seeds,
                                   void *dev_buf, size_t dev_bytes, void *cuda_stream)
{
    if (!dev_buf) return fail(ISING3D_EINVAL, "null device buffer");
    return create(h, L, n_rep, seeds, dev_buf, dev_bytes, cuda_stream);
}

int ising3d_reset(ising3d_t *h)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    return launch_init(h);
}

int ising3d_set_stream(ising3d_t *h, void *cuda_stream)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    h->stream = (cudaStream_t)cuda_stream;
    return ISING3D_OK;
}

int ising3d_set_measure_variant(ising3d_t *h, int variant)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (variant < ISING3D_MEASURE_AUTO || variant > ISING3D_MEASURE_TENSOR)
        return fail(ISING3D_EINVAL, "unknown measurement variant");
    if (variant == ISING3D_MEASURE_TENSOR && !ising::gram_supported(h->L))
        return fail(ISING3D_EINVAL, "the tensor-core measurement needs L to be a multiple of 512");
    h->measure_variant = variant;
    return ISING3D_OK;
}

int ising3d_set_temperature(ising3d_t *h, double T)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (!(T >= 0.0) || !std::isfinite(T)) return fail(ISING3D_EINVAL, "temperature must be finite and >= 0");
    if (T > 0.0 && h->cycle != ISING3D_CYCLE_01)
        return fail(ISING3D_EINVAL, "finite temperature is implemented for the 01 cycle only");
    if (T != h->temperature) {      // other dynamics from here on: the adaptive choice starts over on the dense kernel
        h->active_mode = false;
        h->run_len = 0;
    }
    h->temperature = T;
    if (T > 0.0) {
        // D13: thr[n] = floor(2^32 / (1 + exp((12 - 4n)/T))), fp64, n = antiparallel neighbours
        for (int B = 0; B <= 32; ++B) h->glauber.lut[B] = 0u;
        for (int n = 0; n <= 6; ++n) {
            const double dE = 12.0 - 4.0 * (double)n;
            const double p = 1.0 / (1.0 + std::exp(dE / T));
            const uint64_t thr = (uint64_t)std::floor(p * 4294967296.0);
            for (int B = 0; B <= 32; ++B) h->glauber.lut[B] |= (uint32_t)((thr >> B) & 1u) << n;
        }
    }
    return ISING3D_OK;
}

int ising3d_set_cycle(ising3d_t *h, int cycle)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (cycle < ISING3D_CYCLE_01 || cycle > ISING3D_CYCLE_DOUBLE_CB_MIXED)
        return fail(ISING3D_EINVAL, "unknown cycle");
    if (cycle == ISING3D_CYCLE_DOUBLE_CB_MIXED && h->variant != ISING3D_VARIANT_AUTO &&
        h->variant != ISING3D_VARIANT_GENERIC && h->variant != ISING3D_VARIANT_FUSED2)
        return fail(ISING3D_EINVAL, "the mixed-cycle double checkerboard runs on the fused2 and generic kernels");
    if (cycle != ISING3D_CYCLE_01 && h->temperature > 0.0)
        return fail(ISING3D_EINVAL, "finite temperature is implemented for the 01 cycle only");
    if (cycle != ISING3D_CYCLE_01 && h->variant == ISING3D_VARIANT_FUSED)
        return fail(ISING3D_EINVAL, "the first-generation fused kernel runs the 01 cycle only");
    if (cycle >= ISING3D_CYCLE_DOUBLE_CB && h->variant == ISING3D_VARIANT_FUSED3)
        return fail(ISING3D_EINVAL, "the double checkerboard runs on the resident, fused2 and generic kernels");
    if (cycle >= ISING3D_CYCLE_DOUBLE_CB && h->variant == ISING3D_VARIANT_ACTIVE)
        return fail(ISING3D_EINVAL, "the double checkerboard runs on the resident, fused2 and generic kernels");
    if (cycle != h->cycle) {
        h->active_mode = false;
        h->run_len = 0;
    }
    h->cycle = cycle;
    return ISING3D_OK;
}

int ising3d_init_menger(ising3d_t *h, int k)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    int size = 1;
    for (int i = 0; i < k && size <= 4096; ++i) size *= 3;
    if (k < 0 || k > 7 || size > h->L)
        return fail(ISING3D_EINVAL, "Menger iteration k must satisfy 0 <= k and 3^k <= L");
    const size_t words = h->words_per_replica();
    dim3 grid((unsigned)((words + 255) / 256), (unsigned)h->n_rep);
    ising::init_menger_kernel<<<grid, 256, 0, h->stream>>>(h->state[h->cur], h->d_seeds, h->L, k, size);
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    h->sweep = 0;
    h->state_changed();
    return ISING3D_OK;
}

int ising3d_set_variant(ising3d_t *h, int variant)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (variant < ISING3D_VARIANT_AUTO || variant > ISING3D_VARIANT_ACTIVE)
        return fail(ISING3D_EINVAL, "unknown variant");
    if (variant == ISING3D_VARIANT_ACTIVE && !h->active_ok())
        return fail(ISING3D_EINVAL, "the activity-driven kernel needs L in {256,512,1024,2048,4096}");
    if (variant == ISING3D_VARIANT_ACTIVE && h->cycle >= ISING3D_CYCLE_DOUBLE_CB)
        return fail(ISING3D_EINVAL, "the double checkerboard runs on the resident, fused2 and generic kernels");
    if (h->cycle == ISING3D_CYCLE_DOUBLE_CB_MIXED && variant != ISING3D_VARIANT_AUTO &&
        variant != ISING3D_VARIANT_GENERIC && variant != ISING3D_VARIANT_FUSED2)
        return fail(ISING3D_EINVAL, "the mixed-cycle double checkerboard runs on the fused2 and generic kernels");
    if (variant == ISING3D_VARIANT_FUSED3 && h->cycle >= ISING3D_CYCLE_DOUBLE_CB)
        return fail(ISING3D_EINVAL, "the double checkerboard runs on the resident, fused2 and generic kernels");
    if (variant == ISING3D_VARIANT_FUSED && h->cycle != ISING3D_CYCLE_01)
        return fail(ISING3D_EINVAL, "the first-generation fused kernel runs the 01 cycle only");
    if (variant == ISING3D_VARIANT_FUSED && !h->fused_ok())
        return fail(ISING3D_EINVAL, "fused kernel needs L in {256,512,1024,2048,4096}");
    if (variant == ISING3D_VARIANT_FUSED2 && !h->fused2_ok())
        return fail(ISING3D_EINVAL, "fused2 kernel needs L in {512,1024,1536,2048,4096}");
    if (variant == ISING3D_VARIANT_FUSED3 && !h->fused3_ok())
        return fail(ISING3D_EINVAL, "fused3 kernel needs L in {1024,2048}");
    if (variant == ISING3D_VARIANT_RESIDENT && !h->resident_ok())
        return fail(ISING3D_EINVAL, "resident kernel needs L in {64,128,256} and a cluster that fits");
    h->variant = variant;
    h->active_mode = false;
    h->run_len = 0;
    return ISING3D_OK;
}

int ising3d_set_activity_policy(ising3d_t *h, uint64_t probe_interval, double on_below, double off_above)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (!(on_below >= 0.0) || !(off_above >= on_below) || !(off_above <= 1.0))
        return fail(ISING3D_EINVAL, "need 0 <= on_below <= off_above <= 1");
    h->probe_interval = probe_interval;
    h->active_on = on_below;
    h->active_off = off_above;
    h->active_mode = false;
    h->run_len = 0;
    return ISING3D_OK;
}

int ising3d_activity(ising3d_t *h, uint64_t *awake_groups, double *last_fraction)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (last_fraction) *last_fraction = h->last_activity;
    if (!awake_groups) return ISING3D_OK;
    if (!h->active_ok()) return fail(ISING3D_EINVAL, "activity counts need L in {256,512,1024,2048,4096}");
    // Counting rebuilds the flags from the state: the flags an active run carries are a superset
    // (woken groups not yet evaluated), the rebuilt ones are exact and satisfy the same invariant.
    int rc = build_flags(h);
    if (rc != ISING3D_OK) return rc;
    double frac = 0.0;
    rc = read_activity(h, &frac, awake_groups);
    if (rc != ISING3D_OK) return rc;
    if (last_fraction) *last_fraction = frac;
    return ISING3D_OK;
}

int ising3d_active_stats(ising3d_t *h, uint64_t *evaluated_changed)
{
    if (!h || !evaluated_changed) return fail(ISING3D_EINVAL, "null pointer");
    if (!h->active_ok()) return fail(ISING3D_EINVAL, "the activity-driven kernel needs L in {256,512,1024,2048,4096}");
    std::vector<unsigned long long> host((size_t)h->n_rep * kActStride);
    CUDA_TRY(cudaMemcpyAsync(host.data(), h->d_act, host.size() * 8, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaMemset2DAsync(h->d_act + 2, kActStride * 8, 0, 2 * 8, (size_t)h->n_rep, h->stream));   // [rep][2..3]
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (int rep = 0; rep < h->n_rep; ++rep) {
        evaluated_changed[rep * 2 + 0] = host[rep * kActStride + 2];
        evaluated_changed[rep * 2 + 1] = host[rep * kActStride + 3];
    }
    return ISING3D_OK;
}

int ising3d_set_cluster_size(ising3d_t *h, int cs)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (!ising::resident_supported(h->L))
        return fail(ISING3D_EINVAL, "the resident kernel needs L in {64,128,256}");
    if (cs == 0) {                               // back to the automatic choice
        h->res_planned = false;
        return ISING3D_OK;
    }
    if (cs < 1 || cs > 16 || (cs & (cs - 1)) || h->L / cs < 2 ||
        ising::resident_smem_bytes(h->L, cs) > 200 * 1024)
        return fail(ISING3D_EINVAL, "cluster size must be a power of two <= 16 whose z slab fits shared memory");
    int clusters = 0;
    if (ising::resident_try_size(h->L, cs, h->n_rep, &clusters) != cudaSuccess || clusters < 1) {
        cudaGetLastError();
        return fail(ISING3D_EINVAL, "this device cannot co-schedule a cluster of that size");
    }
    h->res_plan = ising::ResidentPlan{cs, ising::resident_smem_bytes(h->L, cs)};
    h->res_planned = true;
    return ISING3D_OK;
}

int ising3d_sweep(ising3d_t *h, uint64_t n_sweeps)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    if (h->sweep + n_sweeps > 0xFFFFFFFFull || h->sweep + n_sweeps < h->sweep)
        return fail(ISING3D_EINVAL, "sweep counter would pass 2^32-1");
    if (n_sweeps == 0) return ISING3D_OK;
    if (!h->auto_adaptive() && !h->use_active()) h->flags_valid = false;   // kernels that do not keep the flags
    const int rc = h->temperature > 0.0 ? sweep_glauber(h, n_sweeps)
                   : h->use_resident() ? sweep_resident(h, n_sweeps)
                   : h->use_active()   ? sweep_active(h, 0, n_sweeps)
                   : h->auto_adaptive() ? sweep_auto(h, n_sweeps)
                   : h->use_fused2()  ? sweep_fused(h, 0, n_sweeps, true)
                   : h->use_fused() ? sweep_fused(h, 0, n_sweeps, false)
                                    : sweep_generic(h, n_sweeps);
    if (rc != ISING3D_OK) return rc;
    h->sweep += n_sweeps;
    return ISING3D_OK;
}

int ising3d_measure(ising3d_t *h, ising3d_meas_t *out)
{
    if (!h || !out) return fail(ISING3D_EINVAL, "null pointer");
    if (out->L != h->L || out->n_rep != h->n_rep)
        return fail(ISING3D_EINVAL, "measurement record shape does not match the handle");
    if (!out->n_up || !out->n_broken || !out->antipar)
        return fail(ISING3D_EINVAL, "n_up, n_broken and antipar must be provided");
    const int L = h->L, nr = L / 2 + 1, cpr = h->counts_per_replica();
    const uint32_t *st = h->state[h->cur];
    CUDA_TRY(cudaMemsetAsync(h->d_counts, 0, (size_t)h->n_rep * cpr * 8, h->stream));
    {
        const size_t n4 = h->words_per_replica() / 4;
        unsigned gx = (unsigned)std::min<size_t>((n4 + 255) / 256, (size_t)h->sm_count * 8);
        ising::count_up_kernel<<<dim3(gx, h->n_rep), 256, 0, h->stream>>>(
            st, h->d_counts, h->words_per_replica(), cpr);
    }
    if (h->use_gram()) {
        const int rc = measure_gram(h);
        if (rc != ISING3D_OK) return rc;
    } else
    {
        // A_mu(r): persistent CTAs over tiles of C line-word sequences (kernels_measure.cuh)
        const int C = ising::autocorr_tile_sequences(L);
        const int n_tiles = (L * L / 32) / C;
        const size_t smem = ising::autocorr_smem_bytes(L, C);
        if (!h->attr_autocorr) {                    // per device, idempotent; once per handle
            const int max_smem = (int)ising::autocorr_smem_bytes(4096, 8) + 4096;
            CUDA_TRY(cudaFuncSetAttribute(ising::autocorr_kernel<0>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
            CUDA_TRY(cudaFuncSetAttribute(ising::autocorr_kernel<1>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
            CUDA_TRY(cudaFuncSetAttribute(ising::autocorr_kernel<2>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
            h->attr_autocorr = true;
        }
        int gx = std::max(1, (h->sm_count + h->n_rep - 1) / h->n_rep);
        gx = std::min(gx, n_tiles);
        dim3 grid((unsigned)gx, (unsigned)h->n_rep);
        ising::autocorr_kernel<0><<<grid, ising::kAcThreads, smem, h->stream>>>(st, h->d_counts, L, C,
                                                                                n_tiles, cpr);
        ising::autocorr_kernel<1><<<grid, ising::kAcThreads, smem, h->stream>>>(st, h->d_counts, L, C,
                                                                                n_tiles, cpr);
        ising::autocorr_kernel<2><<<grid, ising::kAcThreads, smem, h->stream>>>(st, h->d_counts, L, C,
                                                                                n_tiles, cpr);
        h->launches += 3;
    }
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    std::vector<unsigned long long> host((size_t)h->n_rep * cpr);
    CUDA_TRY(cudaMemcpyAsync(host.data(), h->d_counts, host.size() * 8, cudaMemcpyDeviceToHost,
                             h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    out->sweep = h->sweep;
    for (int rep = 0; rep < h->n_rep; ++rep) {
        const unsigned long long *c = host.data() + (size_t)rep * cpr;
        out->n_up[rep] = c[0];
        uint64_t *a = out->antipar + (size_t)rep * 3 * nr;
        for (int i = 0; i < 3 * nr; ++i) a[i] = c[1 + i];
        out->n_broken[rep] = a[1] + a[nr + 1] + a[2 * nr + 1];
        postprocess(L, out->n_up[rep], a, out->c_intercept,
                    out->C ? out->C + (size_t)rep * nr : nullptr, out->ell ? out->ell + rep : nullptr);
    }
    return ISING3D_OK;
}

int ising3d_measure_static(const uint32_t *dev_words, int L, int n_rep, uint64_t *n_up, uint64_t *antipar,
                           void *cuda_stream)
{
    if (!dev_words || !n_up || !antipar) return fail(ISING3D_EINVAL, "null pointer");
    if (!valid_shape(L, n_rep))
        return fail(ISING3D_EINVAL, "L must be a multiple of 64 in [64, 4096] and n_rep >= 1");
    if ((uintptr_t)dev_words & 15) return fail(ISING3D_EINVAL, "dev_words must be 16-byte aligned");
    const int nr = L / 2 + 1, cpr = 1 + 3 * nr;
    if ((uint64_t)n_rep * (uint64_t)cpr > (uint64_t)ISING3D_STATIC_MAX_COUNTS)
        return fail(ISING3D_EINVAL,
                    "ising3d_measure_static: n_rep * (1 + 3 (L/2+1)) = " + std::to_string((uint64_t)n_rep * cpr) +
                        " counters exceed the static scratch of " + std::to_string(ISING3D_STATIC_MAX_COUNTS) +
                        " (ISING3D_STATIC_MAX_COUNTS); measure fewer replicas per call or use ising3d_measure");
    unsigned long long *counts = nullptr;
    const int rc = static_scratch_for_current_device(&counts);   // first call on a device: set-up
    if (rc != ISING3D_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    int sm_count = 0, dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    // the array keeps the previous call's sums and the kernels only add: clear the part this call uses
    CUDA_TRY(cudaMemsetAsync(counts, 0, (size_t)n_rep * cpr * 8, stream));
    const size_t wpr = (size_t)L * L * L / 32;
    {
        const size_t n4 = wpr / 4;
        const unsigned gx = (unsigned)std::min<size_t>((n4 + 255) / 256, (size_t)sm_count * 8);
        ising::count_up_kernel<<<dim3(gx, n_rep), 256, 0, stream>>>(dev_words, counts, wpr, cpr);
    }
    {
        // same tiling as the popcount branch of ising3d_measure (kernels_measure.cuh)
        const int C = ising::autocorr_tile_sequences(L);
        const int n_tiles = (L * L / 32) / C;
        const size_t smem = ising::autocorr_smem_bytes(L, C);
        int gx = std::max(1, (sm_count + n_rep - 1) / n_rep);
        gx = std::min(gx, n_tiles);
        const dim3 grid((unsigned)gx, (unsigned)n_rep);
        ising::autocorr_kernel<0><<<grid, ising::kAcThreads, smem, stream>>>(dev_words, counts, L, C, n_tiles, cpr);
        ising::autocorr_kernel<1><<<grid, ising::kAcThreads, smem, stream>>>(dev_words, counts, L, C, n_tiles, cpr);
        ising::autocorr_kernel<2><<<grid, ising::kAcThreads, smem, stream>>>(dev_words, counts, L, C, n_tiles, cpr);
    }
    CUDA_TRY(cudaGetLastError());
    // [rep][0] -> n_up[rep], [rep][1 ..] -> antipar[rep][3][nr]: two strided copies straight into the
    // caller's arrays, no staging buffer
    CUDA_TRY(cudaMemcpy2DAsync(n_up, 8, counts, (size_t)cpr * 8, 8, (size_t)n_rep, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaMemcpy2DAsync(antipar, (size_t)3 * nr * 8, counts + 1, (size_t)cpr * 8, (size_t)3 * nr * 8,
                               (size_t)n_rep, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    return ISING3D_OK;
}

int ising3d_measure_radial(ising3d_t *h, ising3d_radial_t *out)
{
    if (!h || !out) return fail(ISING3D_EINVAL, "null pointer");
    if (out->L != h->L || out->n_rep != h->n_rep)
        return fail(ISING3D_EINVAL, "measurement record shape does not match the handle");
    if (!out->corr_sum || !out->shell || !out->C_rad)
        return fail(ISING3D_EINVAL, "corr_sum, shell and C_rad must be provided");
    const int rc = fft_setup(h);
    if (rc != ISING3D_OK) return rc;
    const int L = h->L, H = L / 2 + 1, cpr = h->counts_per_replica();
    const double N = (double)L * L * L;
    if (cufftSetStream(h->plan_fwd, h->stream) != CUFFT_SUCCESS ||
        cufftSetStream(h->plan_inv, h->stream) != CUFFT_SUCCESS)
        return fail(ISING3D_ECUDA, "cufftSetStream failed");
    std::vector<unsigned long long> host((size_t)3 * H + 1);
    const int grid = h->sm_count * 8;
    h->radial_rounding = 0.0;
    out->sweep = h->sweep;
    for (int rep = 0; rep < h->n_rep; ++rep) {
        const uint32_t *st = h->state[h->cur] + (size_t)rep * h->words_per_replica();
        unsigned long long *d_cnt = h->d_counts + (size_t)rep * cpr;
        CUDA_TRY(cudaMemsetAsync(d_cnt, 0, 8, h->stream));
        CUDA_TRY(cudaMemsetAsync(h->d_rad, 0, ((size_t)3 * H + 1) * 8, h->stream));
        ising::count_up_kernel<<<dim3((unsigned)grid, 1), 256, 0, h->stream>>>(st, d_cnt, h->words_per_replica(), cpr);
        ising::unpack_real_kernel<<<grid, 256, 0, h->stream>>>(st, h->fft_buf, L);
        if (cufftExecD2Z(h->plan_fwd, h->fft_buf, reinterpret_cast<cufftDoubleComplex *>(h->fft_buf)) != CUFFT_SUCCESS)
            return fail(ISING3D_ECUDA, "cufftExecD2Z failed");
        ising::power_kernel<<<grid, 256, (size_t)H * 8, h->stream>>>(
            reinterpret_cast<double2 *>(h->fft_buf), reinterpret_cast<double *>(h->d_rad + 2 * H), L);
        if (cufftExecZ2D(h->plan_inv, reinterpret_cast<cufftDoubleComplex *>(h->fft_buf), h->fft_buf) != CUFFT_SUCCESS)
            return fail(ISING3D_ECUDA, "cufftExecZ2D failed");
        ising::radial_kernel<<<grid, 256, (size_t)2 * H * 8, h->stream>>>(h->fft_buf, h->d_rad, h->d_rad + H,
                                                                          h->d_rad + 3 * H, L);
        h->launches += 4;
        CUDA_TRY(cudaGetLastError());
        unsigned long long n_up = 0;
        CUDA_TRY(cudaMemcpyAsync(host.data(), h->d_rad, host.size() * 8, cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaMemcpyAsync(&n_up, d_cnt, 8, cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        {
            double dev;
            std::memcpy(&dev, &host[3 * H], 8);
            h->radial_rounding = std::max(h->radial_rounding, dev);
        }
        // D12 / D9 post-processing in fp64, this order
        const double m = (double)(2 * (int64_t)n_up - (int64_t)N) / N;
        double *C = out->C_rad + (size_t)rep * H;
        for (int b = 0; b < H; ++b) {
            const int64_t ps = (int64_t)host[b];
            out->corr_sum[(size_t)rep * H + b] = ps;
            out->shell[b] = host[H + b];
            C[b] = (double)ps / (N * (double)host[H + b]) - m * m;
            if (out->S_rad) {
                double sv;
                std::memcpy(&sv, &host[2 * H + b], 8);
                out->S_rad[(size_t)rep * H + b] = sv / (N * (double)host[H + b]);
            }
        }
        if (out->ell) {
            out->ell[rep] = std::nan("");
            for (int b = 0; b + 1 < H; ++b)
                if (C[b] >= out->c_intercept && C[b + 1] < out->c_intercept) {
                    out->ell[rep] = (double)b + (C[b] - out->c_intercept) / (C[b] - C[b + 1]);
                    break;
                }
        }
    }
    return ISING3D_OK;
}

int ising3d_radial_rounding(const ising3d_t *h, double *max_distance)
{
    if (!h || !max_distance) return fail(ISING3D_EINVAL, "null pointer");
    *max_distance = h->radial_rounding;
    return ISING3D_OK;
}

int ising3d_release_radial(ising3d_t *h)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    cudaStreamSynchronize(h->stream);
    if (h->plan_fwd) cufftDestroy(h->plan_fwd);
    if (h->plan_inv) cufftDestroy(h->plan_inv);
    if (h->fft_buf) cudaFree(h->fft_buf);
    if (h->fft_work) cudaFree(h->fft_work);
    if (h->d_rad) cudaFree(h->d_rad);
    h->plan_fwd = h->plan_inv = 0;
    h->fft_buf = nullptr;
    h->fft_work = nullptr;
    h->d_rad = nullptr;
    h->fft_ready = false;
    return ISING3D_OK;
}

int ising3d_get_state(ising3d_t *h, uint32_t *words, size_t n_words, uint64_t *sweep)
{
    if (!h || !words) return fail(ISING3D_EINVAL, "null pointer");
    if (n_words != h->words_per_replica() * h->n_rep)
        return fail(ISING3D_EINVAL, "n_words must equal n_rep * L^3/32");
    CUDA_TRY(cudaMemcpyAsync(words, h->state[h->cur], n_words * 4, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (sweep) *sweep = h->sweep;
    return probe_poll(h);
}

int ising3d_set_state(ising3d_t *h, const uint32_t *words, size_t n_words, uint64_t sweep)
{
    if (!h || !words) return fail(ISING3D_EINVAL, "null pointer");
    if (n_words != h->words_per_replica() * h->n_rep)
        return fail(ISING3D_EINVAL, "n_words must equal n_rep * L^3/32");
    if (sweep > 0xFFFFFFFFull) return fail(ISING3D_EINVAL, "sweep counter out of range");
    CUDA_TRY(cudaMemcpyAsync(h->state[h->cur], words, n_words * 4, cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    h->sweep = sweep;
    h->state_changed();
    return ISING3D_OK;
}

int ising3d_get_state_device(ising3d_t *h, uint32_t *dev_words, size_t n_words, uint64_t *sweep)
{
    if (!h || !dev_words) return fail(ISING3D_EINVAL, "null pointer");
    if (n_words != h->words_per_replica() * h->n_rep)
        return fail(ISING3D_EINVAL, "n_words must equal n_rep * L^3/32");
    CUDA_TRY(cudaMemcpyAsync(dev_words, h->state[h->cur], n_words * 4, cudaMemcpyDeviceToDevice,
                             h->stream));
    if (sweep) *sweep = h->sweep;
    return ISING3D_OK;
}

int ising3d_set_state_device(ising3d_t *h, const uint32_t *dev_words, size_t n_words, uint64_t sweep)
{
    if (!h || !dev_words) return fail(ISING3D_EINVAL, "null pointer");
    if (n_words != h->words_per_replica() * h->n_rep)
        return fail(ISING3D_EINVAL, "n_words must equal n_rep * L^3/32");
    if (sweep > 0xFFFFFFFFull) return fail(ISING3D_EINVAL, "sweep counter out of range");
    CUDA_TRY(cudaMemcpyAsync(h->state[h->cur], dev_words, n_words * 4, cudaMemcpyDeviceToDevice,
                             h->stream));
    h->sweep = sweep;
    h->state_changed();
    return ISING3D_OK;
}

int ising3d_L(const ising3d_t *h) { return h ? h->L : 0; }
int ising3d_n_rep(const ising3d_t *h) { return h ? h->n_rep : 0; }
uint64_t ising3d_sweep_count(const ising3d_t *h) { return h ? h->sweep : 0; }
uint64_t ising3d_launch_count(const ising3d_t *h) { return h ? h->launches : 0; }
const char *ising3d_measure_variant_name(const ising3d_t *h)
{
    if (!h) return "none";
    return h->use_gram() ? "tensor" : "popcount";
}

const char *ising3d_variant_name(const ising3d_t *h)
{
    if (!h) return "none";
    if (h->temperature > 0.0) return "glauber";
    if (h->use_active() || (h->auto_adaptive() && h->active_mode && !h->use_resident())) return "active";
    return h->use_resident() ? "resident" : h->use_fused3() ? "fused3" : h->use_fused2() ? "fused2" : h->use_fused() ? "fused" : "generic";
}

int ising3d_cluster_size(const ising3d_t *h)
{
    return (h && h->use_resident()) ? h->res_plan.cs : 0;
}

int ising3d_sync(ising3d_t *h)
{
    if (!h) return fail(ISING3D_EINVAL, "null handle");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return probe_poll(h);        // a probe of the AUTO policy that was in flight has landed: take its result
}

void ising3d_free(ising3d_t *h)
{
    if (!h) return;
    cudaStreamSynchronize(h->stream);
    ising3d_release_radial(h);
    if (h->owns_mem && h->base) cudaFree(h->base);
    if (h->h_probe) cudaFreeHost(h->h_probe);
    if (h->probe_event) cudaEventDestroy(h->probe_event);
    delete h;
}

const char *ising3d_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
