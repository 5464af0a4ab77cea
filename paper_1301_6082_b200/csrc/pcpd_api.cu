// Host side of libpcpd.so: the C ABI declared in include/pcpd.h.
// Argument checking, thresholds (C3), handle state (C7: lattice + sweep counter),
// kernel launches.  No compute happens on the host; there is no CPU fallback.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <mutex>
#include <new>

#include "../../include/pcpd.h"
#include "pcpd_kernels.cuh"

using namespace pcpd;

namespace {

thread_local char g_err[512] = "";
std::atomic<uint64_t> g_launches{0};
// Process-wide state, guarded by g_mu: the allocator pair new handles will use, the number of live handles (the pair
// cannot be swapped under them) and the per-device first-use configuration (the opt-in shared-memory attribute is per
// context).  Everything else a call touches belongs to its handle.
std::mutex g_mu;
pcpd_alloc_fn g_alloc = nullptr;
pcpd_free_fn g_free = nullptr;
uint64_t g_live = 0;
bool g_configured[64] = {};

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

int cuda_fail(cudaError_t e, const char *what)
{
    return fail(PCPD_ERR_DEVICE, "%s: %s", what, cudaGetErrorString(e));
}

// device memory through the allocator pair the handle was created with (NULL pair: cudaMalloc / cudaFree)
struct Allocator {
    pcpd_alloc_fn alloc;
    pcpd_free_fn release;
};

void *dev_alloc(const Allocator &a, size_t bytes, cudaStream_t s)
{
    if (a.alloc) return a.alloc(bytes, (void *)s);
    void *p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    return p;
}

void dev_free(const Allocator &a, void *p)
{
    if (!p) return;
    if (a.release) a.release(p);
    else cudaFree(p);
}

// T = floor(q * 2^32) in double arithmetic (C3); q in [0,1].
uint64_t threshold_of(double q) { return (uint64_t)std::floor(std::ldexp(q, 32)); }

Threshold make_threshold(uint64_t T)
{
    Threshold th{};
    th.all = (T >= (1ull << 32)) ? 1u : 0u;
    th.T32 = th.all ? 0u : (uint32_t)T;
    th.nplanes = (th.all || T == 0) ? 0u : 32u - (uint32_t)__builtin_ctz((uint32_t)T);
    return th;
}

}  // namespace

struct pcpd_s {
    uint64_t L, R, W;
    double d, p;
    uint64_t seed;
    int variant;
    uint32_t Ts, D, A;
    uint64_t word_offset;
    uint64_t Td, Tp;
    uint64_t sweep;
    bool force_block;  // test hook (env PCPD_FORCE_BLOCK_KERNEL=1 at create): run the generic block kernel
    bool invalid;      // a pipelined pcpd_step_from_host failed part-way: the lattice is undefined until set_lattice / init
    int connected;     // PCPD_VARIANT_CONNECTED
    Allocator mem;     // the allocator pair in force when the handle was created
    uint32_t *thr;     // device, per-word thresholds [W][4] (pcpd_create_scan), else NULL
    uint64_t *lat;     // device, column-major [W][L]
    uint32_t *counts;  // device, uint32[R]
    cudaStream_t stream;
    SweepParams P;
    JitSlot jit;       // threshold-specialised sweep kernel (jit.cu); mode from env PCPD_JIT at create
    SplitSlot split;   // small / mid-size problems: column_kernel (sweep_warp.cu); env PCPD_SPLIT
    // pcpd_step_from_host: copy stream and events, created on first use and kept for the life of the handle
    cudaStream_t copy_stream;
    cudaEvent_t copy_start;
    cudaEvent_t *chunk_ev;
    uint32_t n_chunk_ev;
    int device;        // the device that was current at create (pcpd_run_series_static checks it)
};

static void release_handle(pcpd_s *h)   // frees everything the handle owns (partially constructed handles too)
{
    if (h->copy_stream) {
        cudaStreamSynchronize(h->copy_stream);
        cudaStreamDestroy(h->copy_stream);
    }
    if (h->copy_start) cudaEventDestroy(h->copy_start);
    for (uint32_t c = 0; c < h->n_chunk_ev; ++c)
        if (h->chunk_ev[c]) cudaEventDestroy(h->chunk_ev[c]);
    delete[] h->chunk_ev;
    dev_free(h->mem, h->thr);
    dev_free(h->mem, h->lat);
    dev_free(h->mem, h->counts);
    delete h;
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_live) --g_live;
}

extern "C" {

const char *pcpd_last_error(void) { return g_err; }
uint64_t pcpd_launch_count(void) { return g_launches.load(); }

int pcpd_set_allocator(pcpd_alloc_fn alloc, pcpd_free_fn release)
{
    if ((alloc == nullptr) != (release == nullptr)) return fail(PCPD_ERR_ARG, "set_allocator: give both or neither");
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_live && (alloc != g_alloc || release != g_free))
        return fail(PCPD_ERR_ARG, "set_allocator: %llu handle(s) are alive; destroy them first", (unsigned long long)g_live);
    g_alloc = alloc;
    g_free = release;
    return PCPD_OK;
}

pcpd_t *pcpd_create_ex(uint64_t L, uint64_t n_replicas, double d, double p, uint64_t seed, int variant, uint32_t Ts,
                       uint32_t D, uint32_t A, uint64_t word_offset)
{
    const int pmask_paper = (variant & PCPD_VARIANT_PMASK_PAPER) ? 1 : 0;
    const int connected = (variant & PCPD_VARIANT_CONNECTED) ? 1 : 0;
    const int pmask_code = (variant & PCPD_VARIANT_PMASK_BOUND_3_4) >> 10;   // 0: b = 1/4, 1: 1/2, 2: 1, 3: 3/4
    variant &= ~(PCPD_VARIANT_PMASK_PAPER | PCPD_VARIANT_CONNECTED | PCPD_VARIANT_PMASK_BOUND_3_4);
    if (pmask_code && !pmask_paper) {
        fail(PCPD_ERR_ARG, "the PCPD_VARIANT_PMASK_BOUND_* bits need PCPD_VARIANT_PMASK_PAPER");
        return nullptr;
    }
    if (variant != PCPD_VARIANT_PCPD && variant != PCPD_VARIANT_TCPD && variant != PCPD_VARIANT_QCPD &&
        variant != PCPD_VARIANT_CPD) {
        fail(PCPD_ERR_ARG, "unknown variant %d", variant);
        return nullptr;
    }
    const uint32_t Rr = variant == PCPD_VARIANT_CPD ? 1u : 2u + (uint32_t)variant;
    if (n_replicas == 0 || n_replicas % 64) {
        fail(PCPD_ERR_ARG, "n_replicas must be a positive multiple of 64");
        return nullptr;
    }
    const uint64_t W = n_replicas / 64;
    if (!(d >= 0.0 && d <= 1.0) || !(p >= 0.0 && p <= 1.0)) {
        fail(PCPD_ERR_ARG, "d and p must lie in [0,1]");
        return nullptr;
    }
    static const double kBound[4] = {0.25, 0.5, 1.0, 0.75};
    if (pmask_paper && !(p < kBound[pmask_code])) {
        fail(PCPD_ERR_ARG, "the paper's annihilation mask needs p < b = %g (its decorrelation bound; default 1/4)", kBound[pmask_code]);
        return nullptr;
    }
    if (L == 0 || L > (1ull << 31) || word_offset + W >= (1ull << 32)) {
        fail(PCPD_ERR_ARG, "L must be <= 2^31 and word_offset + W < 2^32 (32-bit counter fields and site indices)");
        return nullptr;
    }
    if (D == 0 || A == 0 || Ts == 0 || D % A) {
        fail(PCPD_ERR_ARG, "schedule: need A | D, all non-zero");
        return nullptr;
    }
    if (D < 2 * Rr + 3) {
        fail(PCPD_ERR_ARG, "schedule: D must be >= %u for this variant", 2 * Rr + 3);
        return nullptr;
    }
    if (L < D || L % D) {
        fail(PCPD_ERR_ARG, "L must be a multiple of the domain length D = %u", D);
        return nullptr;
    }
    if (Ts > L) Ts = (uint32_t)L;  // clamp
    if (Ts % D || L % Ts) {
        fail(PCPD_ERR_ARG, "schedule: need D | T_s | L (T_s = %u, D = %u)", Ts, D);
        return nullptr;
    }
    if (D / A > MAX_SUBSTEPS) {
        fail(PCPD_ERR_ARG, "schedule: D / A must be <= %u", MAX_SUBSTEPS);
        return nullptr;
    }
    // Physical layout: column-major [W][L]: a tile column is one contiguous run of T_s words, which is
    // what the warp-per-(tile, column) sweep kernel loads.
    if (pmask_paper && !sweep_warp_supported(Ts, D)) {
        fail(PCPD_ERR_ARG, "the paper's annihilation mask needs at most 32 domains per tile (T_s / D <= 32)");
        return nullptr;
    }
    if (!sweep_warp_supported(Ts, D) && (sweep_smem_bytes(Ts) > 200 * 1024 || (uint64_t)(Ts / D) > 1024)) {
        fail(PCPD_ERR_ARG, "schedule: tile of %u sites does not fit one thread block", Ts);
        return nullptr;
    }
    if (W > 65535) {
        fail(PCPD_ERR_ARG, "too many word columns for one handle (W > 65535): shard by word_offset");
        return nullptr;
    }

    int dev = 0;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) {
        cuda_fail(e, "no CUDA device");
        return nullptr;
    }
    if (prop.major != 10) {
        fail(PCPD_ERR_DEVICE, "device is sm_%d%d; this library is built for sm_100a only", prop.major, prop.minor);
        return nullptr;
    }
    if (dev < 0 || dev >= 64) {
        fail(PCPD_ERR_DEVICE, "device index %d out of range", dev);
        return nullptr;
    }
    pcpd_s *h = new (std::nothrow) pcpd_s();
    if (!h) {
        fail(PCPD_ERR_ALLOC, "host allocation failed");
        return nullptr;
    }
    {
        // first use of a device configures the kernels (opt-in shared memory); serialised, as is the snapshot of
        // the allocator pair this handle will allocate and free with
        std::lock_guard<std::mutex> lk(g_mu);
        if (!g_configured[dev]) {
            const int rc = configure_kernels();
            if (rc != 0) {
                delete h;
                cuda_fail((cudaError_t)rc, "cudaFuncSetAttribute");
                return nullptr;
            }
            g_configured[dev] = true;
        }
        h->mem = Allocator{g_alloc, g_free};
        ++g_live;
    }
    h->L = L; h->R = n_replicas; h->W = W; h->d = d; h->p = p; h->seed = seed; h->variant = variant;
    h->Ts = Ts; h->D = D; h->A = A; h->word_offset = word_offset; h->sweep = 0;
    h->Td = threshold_of(d); h->Tp = threshold_of(p);
    h->invalid = false;
    h->device = dev;
    h->connected = connected;
    h->copy_stream = nullptr; h->copy_start = nullptr; h->chunk_ev = nullptr; h->n_chunk_ev = 0;
    {
        const char *fb = getenv("PCPD_FORCE_BLOCK_KERNEL");
        h->force_block = fb && fb[0] == '1' && !pmask_paper && (uint64_t)(Ts / D) <= 1024 &&
                         sweep_smem_bytes(Ts) <= 200 * 1024;
    }
    {
        const char *jm = getenv("PCPD_JIT");  // unset / "1": auto (large problems); "0": off; "force": every size
        h->jit.mode = !jm ? 1 : !strcmp(jm, "0") ? 0 : !strcmp(jm, "force") ? 2 : 1;
        h->jit.state = 0;
        h->jit.kernel = nullptr;
        h->jit.wpb = 0;
    }
    memset(&h->split, 0, sizeof h->split);
    h->stream = nullptr;
    h->thr = nullptr;
    h->lat = (uint64_t *)dev_alloc(h->mem, 8 * L * W, h->stream);
    h->counts = (uint32_t *)dev_alloc(h->mem, 4 * n_replicas, h->stream);
    if (!h->lat || !h->counts) {
        release_handle(h);
        fail(PCPD_ERR_ALLOC, "device allocation of %llu bytes failed", (unsigned long long)(8 * L * W));
        return nullptr;
    }
    SweepParams &P = h->P;
    memset(&P, 0, sizeof P);
    P.lat = h->lat; P.L = (uint32_t)L; P.W = (uint32_t)W; P.Ts = Ts; P.D = D; P.A = A; P.S = D / A; P.n = Ts / D;
    P.word_offset = (uint32_t)word_offset;
    P.thd = make_threshold(h->Td);
    P.thp = make_threshold(h->Tp);
    P.rk = make_round_keys(seed);
    P.connected = (uint32_t)connected;
    P.pmask_paper = (uint32_t)pmask_paper;
    // gate threshold floor((p/b) * 2^32) with p/b formed as the paper writes it: 4p, 2p, p, 4p/3 (< 2^32 because p < b)
    const double gate_q = pmask_code == 0 ? 4.0 * p : pmask_code == 1 ? 2.0 * p : pmask_code == 2 ? p : 4.0 * p / 3.0;
    P.T4p = pmask_paper ? (uint32_t)threshold_of(gate_q) : 0u;
    P.pmask_code = (uint32_t)pmask_code;
    for (int k = 0; k < 32; ++k) {
        P.tdm[k] = ((P.thd.T32 >> (31 - k)) & 1u) ? 0xffffffffu : 0u;
        P.tpm[k] = ((P.thp.T32 >> (31 - k)) & 1u) ? 0xffffffffu : 0u;
    }
    auto tbit = [](uint32_t T32, int k) -> int32_t { return (k < 0 || k > 31) ? 0 : (int32_t)((T32 >> (31 - k)) & 1u); };
    for (int k = 0; k < 34; ++k) {
        P.sd[k] = tbit(P.thd.T32, k) - tbit(P.thd.T32, k - 1);
        P.sp[k] = tbit(P.thp.T32, k) - tbit(P.thp.T32, k - 1);
    }
    for (int M = 0; M < 18; ++M) {
        P.cld[M] = -tbit(P.thd.T32, 2 * M - 1);
        P.clp[M] = -tbit(P.thp.T32, 2 * M - 1);
    }
    {
        // Small and mid-size problems - too few tile columns to fill the GPU with one warp each - run column_kernel
        // (column_device.cuh): one block per tile column, producer warps computing the state-independent part of every
        // attempt, two update warps (one per 32-bit half of the replica lanes) applying them in order.  Measured on B200
        // at L = 65536, generic thresholds, per sweep (fused warp kernel -> column kernel): 128 columns 75 -> 18.6 us,
        // 256: 76 -> 31 us, 512: 76 -> 57 us, 768: 91 -> 82 us; the limit (column_task_limit, sweep_warp.cu) is lower for
        // thresholds that need few Philox blocks.
        // PCPD_SPLIT: unset / "1" auto; "0" never; "column" at every size (test hook).
        const char *sm = getenv("PCPD_SPLIT");
        const int mode = !sm ? 1 : !strcmp(sm, "0") ? 0 : !strcmp(sm, "column") ? 2 : 1;
        const uint64_t ntasks = (L / Ts) * W;
        if ((mode == 2 || (mode == 1 && ntasks <= column_task_limit(P))) && column_supported(Ts, D) && !h->force_block)
            h->split.column_mode = 1;
    }
    g_err[0] = 0;
    return h;
}

pcpd_t *pcpd_create(uint64_t L, uint64_t n_replicas, double d, double p, uint64_t seed, int variant)
{
    return pcpd_create_ex(L, n_replicas, d, p, seed, variant, PCPD_DEFAULT_TS, PCPD_DEFAULT_D, PCPD_DEFAULT_A, 0);
}

pcpd_t *pcpd_create_scan(uint64_t L, uint64_t n_replicas, const double *d_w, const double *p_w, uint64_t seed,
                         int variant, uint32_t Ts, uint32_t D, uint32_t A, uint64_t word_offset)
{
    if (!d_w || !p_w) {
        fail(PCPD_ERR_ARG, "create_scan: NULL probability array");
        return nullptr;
    }
    if (variant & PCPD_VARIANT_PMASK_PAPER) {
        fail(PCPD_ERR_ARG, "create_scan: the paper's annihilation mask is not available with per-word probabilities");
        return nullptr;
    }
    if (n_replicas == 0 || n_replicas % 64) {
        fail(PCPD_ERR_ARG, "n_replicas must be a positive multiple of 64");
        return nullptr;
    }
    const uint64_t W = n_replicas / 64;
    for (uint64_t w = 0; w < W; ++w)
        if (!(d_w[w] >= 0.0 && d_w[w] <= 1.0) || !(p_w[w] >= 0.0 && p_w[w] <= 1.0)) {
            fail(PCPD_ERR_ARG, "create_scan: d_w[%llu] / p_w[%llu] must lie in [0,1]", (unsigned long long)w,
                 (unsigned long long)w);
            return nullptr;
        }
    // per-word thresholds exist in the warp-per-tile-column kernel only: the schedule must be one it can run
    if (Ts == 0 || D == 0 || !sweep_warp_supported((uint32_t)(Ts > L ? L : Ts), D)) {
        fail(PCPD_ERR_ARG, "create_scan needs at most 32 domains per tile (T_s / D <= 32) and a tile column of at most "
                           "200 KiB (T_s <= 25598)");
        return nullptr;
    }
    pcpd_t *h = pcpd_create_ex(L, n_replicas, d_w[0], p_w[0], seed, variant, Ts, D, A, word_offset);
    if (!h) return nullptr;
    uint32_t *host = new (std::nothrow) uint32_t[4 * W];
    h->thr = (uint32_t *)dev_alloc(h->mem, 16 * W, h->stream);
    if (!host || !h->thr) {
        delete[] host;
        pcpd_destroy(h);
        fail(PCPD_ERR_ALLOC, "create_scan: allocation of the threshold table failed");
        return nullptr;
    }
    for (uint64_t w = 0; w < W; ++w) {
        const uint64_t Td = threshold_of(d_w[w]), Tp = threshold_of(p_w[w]);
        host[4 * w + 0] = (Td >> 32) ? 0u : (uint32_t)Td;
        host[4 * w + 1] = (Tp >> 32) ? 0u : (uint32_t)Tp;
        host[4 * w + 2] = ((Td >> 32) ? 1u : 0u) | ((Tp >> 32) ? 2u : 0u);
        host[4 * w + 3] = 0u;
    }
    const cudaError_t e = cudaMemcpy(h->thr, host, 16 * W, cudaMemcpyHostToDevice);
    delete[] host;
    if (e != cudaSuccess) {
        pcpd_destroy(h);
        cuda_fail(e, "create_scan: upload of the threshold table");
        return nullptr;
    }
    h->P.thr_dev = h->thr;
    h->force_block = false;
    h->split.column_mode = 0;   // per-word thresholds run the fused kernel
    return h;
}

void pcpd_destroy(pcpd_t *h)
{
    if (!h) return;
    cudaStreamSynchronize(h->stream);
    release_handle(h);
}

int pcpd_set_stream(pcpd_t *h, void *cuda_stream)
{
    if (!h) return fail(PCPD_ERR_ARG, "null handle");
    h->stream = (cudaStream_t)cuda_stream;
    return PCPD_OK;
}

static const char kInvalidMsg[] =
    "the handle's lattice is undefined (a pipelined pcpd_step_from_host failed part-way): call pcpd_set_lattice or pcpd_init";

static int check_launch(const char *what)
{
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, what);
    return PCPD_OK;
}

int pcpd_init(pcpd_t *h, int mode)
{
    if (!h) return fail(PCPD_ERR_ARG, "null handle");
    if (mode < 0 || mode > 2) return fail(PCPD_ERR_ARG, "unknown init mode %d", mode);
    g_launches += launch_init(h->lat, (uint32_t)h->L, (uint32_t)h->W, (uint32_t)h->word_offset, mode, h->P.rk, h->stream);
    h->sweep = 0;
    h->invalid = false;
    return check_launch("init kernel");
}

int pcpd_run(pcpd_t *h, uint64_t n_sweeps)
{
    if (!h) return fail(PCPD_ERR_ARG, "null handle");
    if (h->invalid) return fail(PCPD_ERR_DEVICE, "%s", kInvalidMsg);
    if (h->sweep + n_sweeps > 0xffffffffull) return fail(PCPD_ERR_RANGE, "sweep counter would exceed 2^32-1");
    for (uint64_t it = 0; it < n_sweeps; ++it) {
        h->P.t = (uint32_t)h->sweep;
        g_launches += launch_sweep(h->P, h->variant, h->force_block, h->stream, &h->jit, &h->split);
        h->sweep += 1;
    }
    return check_launch("sweep kernel");
}

static int density_impl(pcpd_t *h, uint32_t *out, int pairs)
{
    if (!h || !out) return fail(PCPD_ERR_ARG, "null argument");
    if (h->invalid) return fail(PCPD_ERR_DEVICE, "%s", kInvalidMsg);
    cudaError_t e = cudaMemsetAsync(h->counts, 0, 4 * h->R, h->stream);
    if (e != cudaSuccess) return cuda_fail(e, "memset");
    g_launches += launch_density(h->lat, (uint32_t)h->L, (uint32_t)h->W, pairs, h->connected, h->counts, h->stream);
    int rc = check_launch("density kernel");
    if (rc) return rc;
    e = cudaMemcpyAsync(out, h->counts, 4 * h->R, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(e, "density read-back");
    return PCPD_OK;
}

int pcpd_density(pcpd_t *h, uint32_t *out_counts) { return density_impl(h, out_counts, 0); }
int pcpd_pair_density(pcpd_t *h, uint32_t *out_pairs) { return density_impl(h, out_pairs, 1); }

int pcpd_run_series(pcpd_t *h, const uint64_t *times, uint64_t n_times, uint32_t *out_counts, uint32_t *out_pairs)
{
    if (!h || !times || n_times == 0 || (!out_counts && !out_pairs)) return fail(PCPD_ERR_ARG, "run_series: null argument");
    for (uint64_t k = 0; k < n_times; ++k) {
        if (times[k] < (k ? times[k - 1] : h->sweep)) return fail(PCPD_ERR_ARG, "run_series: times must ascend from the current sweep");
        if (times[k] > 0xffffffffull) return fail(PCPD_ERR_RANGE, "sweep counter would exceed 2^32-1");
    }
    const int nobs = (out_counts ? 1 : 0) + (out_pairs ? 1 : 0);
    const size_t row = 4 * h->R, bytes = row * n_times * nobs;
    uint32_t *series = (uint32_t *)dev_alloc(h->mem, bytes, h->stream);
    if (!series) return fail(PCPD_ERR_ALLOC, "run_series: allocation of %llu bytes failed", (unsigned long long)bytes);
    cudaError_t e = cudaMemsetAsync(series, 0, bytes, h->stream);
    int rc = PCPD_OK;
    for (uint64_t k = 0; e == cudaSuccess && rc == PCPD_OK && k < n_times; ++k) {
        rc = pcpd_run(h, times[k] - h->sweep);
        if (rc != PCPD_OK) break;
        uint32_t *dst = series + (size_t)k * h->R * nobs;   // record k: [counts][pairs]
        if (out_counts) g_launches += launch_density(h->lat, (uint32_t)h->L, (uint32_t)h->W, 0, 0, dst, h->stream);
        if (out_pairs)
            g_launches += launch_density(h->lat, (uint32_t)h->L, (uint32_t)h->W, 1, h->connected, dst + (out_counts ? h->R : 0),
                                         h->stream);
        rc = check_launch("density kernel");
    }
    // ONE read-back and ONE synchronisation for the whole series
    if (e == cudaSuccess && rc == PCPD_OK) {
        if (nobs == 1) {
            e = cudaMemcpyAsync(out_counts ? out_counts : out_pairs, series, bytes, cudaMemcpyDeviceToHost, h->stream);
        } else {
            e = cudaMemcpy2DAsync(out_counts, row, series, 2 * row, row, n_times, cudaMemcpyDeviceToHost, h->stream);
            if (e == cudaSuccess)
                e = cudaMemcpy2DAsync(out_pairs, row, series + h->R, 2 * row, row, n_times, cudaMemcpyDeviceToHost, h->stream);
        }
    }
    const cudaError_t es = cudaStreamSynchronize(h->stream);
    dev_free(h->mem, series);
    if (rc != PCPD_OK) return rc;
    if (e == cudaSuccess) e = es;
    if (e != cudaSuccess) return cuda_fail(e, "run_series");
    return PCPD_OK;
}

// ---- pcpd_run_series_static: the record buffer of pcpd_run_series as a fixed array in the library image -------------
// In host code the array's NAME is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current (g_series_ptr, guarded by g_mu).
static __device__ __align__(256) uint32_t g_series_scratch[PCPD_STATIC_SERIES_MAX_COUNTS];
static uint32_t *g_series_ptr[64] = {};

// would the handle's next sweep compile its run-time specialised kernel (jit.cu: NVRTC + module load, which allocate)?
// Mirrors the dispatch of launch_sweep / launch_sweep_warp.
static bool next_sweep_would_compile(const pcpd_s *h)
{
    if (h->jit.state != 0 || !h->jit.mode || h->thr || h->force_block) return false;
    if (!sweep_warp_supported(h->Ts, h->D)) return false;
    if (h->jit.mode != 2 && h->split.column_mode) return false;
    if (h->P.thd.all || h->P.thp.all) return false;
    return h->jit.mode == 2 || (h->L / h->Ts) * h->W > column_task_limit(h->P);
}

int pcpd_run_series_static(pcpd_t *h, const uint64_t *times, uint64_t n_times, uint32_t *out_counts, uint32_t *out_pairs)
{
    if (!h || !times || n_times == 0 || (!out_counts && !out_pairs)) return fail(PCPD_ERR_ARG, "run_series_static: null argument");
    for (uint64_t k = 0; k < n_times; ++k) {
        if (times[k] < (k ? times[k - 1] : h->sweep))
            return fail(PCPD_ERR_ARG, "run_series_static: times must ascend from the current sweep");
        if (times[k] > 0xffffffffull) return fail(PCPD_ERR_RANGE, "sweep counter would exceed 2^32-1");
    }
    const uint64_t nobs = (out_counts ? 1 : 0) + (out_pairs ? 1 : 0);
    if (n_times > PCPD_STATIC_SERIES_MAX_COUNTS || n_times * h->R * nobs > PCPD_STATIC_SERIES_MAX_COUNTS)
        return fail(PCPD_ERR_ARG,
                    "run_series_static: %llu records x %llu replicas x %llu observable(s) exceed the maximum of %u counts "
                    "of the static buffer: split the series or use pcpd_run_series",
                    (unsigned long long)n_times, (unsigned long long)h->R, (unsigned long long)nobs, PCPD_STATIC_SERIES_MAX_COUNTS);
    if (times[n_times - 1] > h->sweep && next_sweep_would_compile(h))
        return fail(PCPD_ERR_ARG, "run_series_static: the handle's first sweep compiles its run-time specialised kernel, which "
                                  "allocates: run one sweep with pcpd_run first");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "run_series_static: cudaGetDevice");
    if (dev != h->device || dev < 0 || dev >= 64)
        return fail(PCPD_ERR_DEVICE, "run_series_static: current device %d is not the handle's device %d", dev, h->device);
    uint32_t *series = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        if (!g_series_ptr[dev]) {
            uint32_t *ptr = nullptr;
            e = cudaGetSymbolAddress((void **)&ptr, g_series_scratch);
            if (e != cudaSuccess || !ptr) return cuda_fail(e, "run_series_static: cudaGetSymbolAddress");
            g_series_ptr[dev] = ptr;
        }
        series = g_series_ptr[dev];
    }
    const size_t row = 4 * h->R, bytes = row * n_times * nobs;
    // the density kernel accumulates with atomics and the buffer holds the last call's records: clear what is used
    e = cudaMemsetAsync(series, 0, bytes, h->stream);
    int rc = PCPD_OK;
    for (uint64_t k = 0; e == cudaSuccess && rc == PCPD_OK && k < n_times; ++k) {
        rc = pcpd_run(h, times[k] - h->sweep);
        if (rc != PCPD_OK) break;
        uint32_t *dst = series + (size_t)k * h->R * nobs;   // record k: [counts][pairs]
        if (out_counts) g_launches += launch_density(h->lat, (uint32_t)h->L, (uint32_t)h->W, 0, 0, dst, h->stream);
        if (out_pairs)
            g_launches += launch_density(h->lat, (uint32_t)h->L, (uint32_t)h->W, 1, h->connected, dst + (out_counts ? h->R : 0),
                                         h->stream);
        rc = check_launch("density kernel");
    }
    if (e == cudaSuccess && rc == PCPD_OK) {
        if (nobs == 1) {
            e = cudaMemcpyAsync(out_counts ? out_counts : out_pairs, series, bytes, cudaMemcpyDeviceToHost, h->stream);
        } else {
            e = cudaMemcpy2DAsync(out_counts, row, series, 2 * row, row, n_times, cudaMemcpyDeviceToHost, h->stream);
            if (e == cudaSuccess)
                e = cudaMemcpy2DAsync(out_pairs, row, series + h->R, 2 * row, row, n_times, cudaMemcpyDeviceToHost, h->stream);
        }
    }
    const cudaError_t es = cudaStreamSynchronize(h->stream);
    if (rc != PCPD_OK) return rc;
    if (e == cudaSuccess) e = es;
    if (e != cudaSuccess) return cuda_fail(e, "run_series_static");
    return PCPD_OK;
}

int pcpd_delta_eff(const uint64_t *times, uint64_t n_times, const uint32_t *series, uint64_t n_replicas, uint64_t L,
                   uint32_t half_window, double *out_rho, double *out_delta)
{
    if (!times || !series || !out_rho || !out_delta || n_times == 0 || n_replicas == 0 || L == 0 || half_window == 0)
        return fail(PCPD_ERR_ARG, "delta_eff: null or zero argument");
    for (uint64_t k = 1; k < n_times; ++k)
        if (times[k] < times[k - 1]) return fail(PCPD_ERR_ARG, "delta_eff: times must ascend");
    for (uint64_t k = 0; k < n_times; ++k) {
        uint64_t sum = 0;   // exact: at most 2^32 replicas x counts below 2^32
        for (uint64_t r = 0; r < n_replicas; ++r) sum += series[k * n_replicas + r];
        out_rho[k] = (double)sum / ((double)n_replicas * (double)L);
    }
    const uint64_t m = half_window;
    for (uint64_t k = 0; k < n_times; ++k) {
        double v = std::nan("");
        if (k >= m && k + m < n_times) {
            const uint64_t t0 = times[k - m], t1 = times[k + m];
            const double r0 = out_rho[k - m], r1 = out_rho[k + m];
            if (t0 > 0 && t1 > t0 && r0 > 0.0 && r1 > 0.0) v = -std::log(r1 / r0) / std::log((double)t1 / (double)t0);
        }
        out_delta[k] = v;
    }
    return PCPD_OK;
}

int pcpd_get_lattice(pcpd_t *h, uint64_t *out_words)
{
    if (!h || !out_words) return fail(PCPD_ERR_ARG, "null argument");
    if (h->invalid) return fail(PCPD_ERR_DEVICE, "%s", kInvalidMsg);
    const size_t bytes = 8 * h->L * h->W;
    cudaError_t e;
    if (h->W == 1) {  // a single column: device layout == canonical
        e = cudaMemcpyAsync(out_words, h->lat, bytes, cudaMemcpyDeviceToHost, h->stream);
    } else {
        uint64_t *tmp = (uint64_t *)dev_alloc(h->mem, bytes, h->stream);
        if (!tmp) return fail(PCPD_ERR_ALLOC, "staging allocation failed");
        g_launches += launch_transpose(h->lat, tmp, (uint32_t)h->L, (uint32_t)h->W, 0, h->stream);
        e = cudaMemcpyAsync(out_words, tmp, bytes, cudaMemcpyDeviceToHost, h->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
        dev_free(h->mem, tmp);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(e, "get_lattice");
    return check_launch("transpose kernel");
}

int pcpd_set_lattice(pcpd_t *h, const uint64_t *in_words)
{
    if (!h || !in_words) return fail(PCPD_ERR_ARG, "null argument");
    const size_t bytes = 8 * h->L * h->W;
    cudaError_t e;
    if (h->W == 1) {
        e = cudaMemcpyAsync(h->lat, in_words, bytes, cudaMemcpyHostToDevice, h->stream);
    } else {
        uint64_t *tmp = (uint64_t *)dev_alloc(h->mem, bytes, h->stream);
        if (!tmp) return fail(PCPD_ERR_ALLOC, "staging allocation failed");
        e = cudaMemcpyAsync(tmp, in_words, bytes, cudaMemcpyHostToDevice, h->stream);
        g_launches += launch_transpose(tmp, h->lat, (uint32_t)h->L, (uint32_t)h->W, 1, h->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
        dev_free(h->mem, tmp);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(e, "set_lattice");
    const int rc = check_launch("transpose kernel");
    if (rc == PCPD_OK) h->invalid = false;
    return rc;
}

// Column chunk of the pipelined step: 8 word columns (64-byte rows of the canonical host layout) when the handle has
// at least 16 columns and a chunk is large enough to fill the GPU; otherwise no pipelining.
static uint32_t step_chunk_columns(const pcpd_t *h)
{
    const char *e = getenv("PCPD_STEP_CHUNK");   // tuning hook: columns per chunk (0 = no pipelining)
    if (e) {
        const long v = atol(e);
        return v <= 0 || (uint64_t)v >= h->W ? (uint32_t)h->W : (uint32_t)v;
    }
    if (h->W < 16 || (h->L / h->Ts) * 8 < 148ull * 14) return (uint32_t)h->W;
    return 8u;
}

// copy stream and per-chunk events of the pipelined steps: created on first use, kept for the life of the handle
static int ensure_copy_resources(pcpd_t *h, uint32_t nchunks)
{
    cudaError_t e = cudaSuccess;
    if (!h->copy_stream) e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess && !h->copy_start) e = cudaEventCreateWithFlags(&h->copy_start, cudaEventDisableTiming);
    if (e == cudaSuccess && h->n_chunk_ev < nchunks) {
        cudaEvent_t *ev = new (std::nothrow) cudaEvent_t[nchunks]();
        if (!ev) return fail(PCPD_ERR_ALLOC, "host allocation failed");
        for (uint32_t c = 0; c < h->n_chunk_ev; ++c) ev[c] = h->chunk_ev[c];
        delete[] h->chunk_ev;
        h->chunk_ev = ev;
        for (; e == cudaSuccess && h->n_chunk_ev < nchunks; ++h->n_chunk_ev)
            e = cudaEventCreateWithFlags(&h->chunk_ev[h->n_chunk_ev], cudaEventDisableTiming);
        if (e != cudaSuccess) --h->n_chunk_ev;   // (the slot of the failed creation holds nothing)
    }
    if (e != cudaSuccess) return cuda_fail(e, "step_from_host: copy stream / events");
    return PCPD_OK;
}

// Column-major host buffer (the device's own layout): chunks of columns are contiguous, so every chunk is ONE plain copy
// straight into the lattice - no staging buffer, no transpose - at the full host-to-device rate.
int pcpd_step_from_host_columns(pcpd_t *h, const uint64_t *in_columns, uint64_t n_sweeps, uint32_t *out_counts)
{
    if (!h || !in_columns) return fail(PCPD_ERR_ARG, "null argument");
    if (h->sweep + n_sweeps > 0xffffffffull) return fail(PCPD_ERR_RANGE, "sweep counter would exceed 2^32-1");
    const uint32_t L = (uint32_t)h->L, W = (uint32_t)h->W;
    // chunk unit: the most columns that still fit two full waves of warps (2 x 148 SMs x 14 warps) - a launch of 2.2
    // waves costs three wave-times, one of 1.98 two - so that the first, exposed copy is short and no launch ends in a
    // nearly empty wave; handles too small for two such chunks copy the whole lattice first
    uint32_t cw = W;
    if (const char *e = getenv("PCPD_STEP_CHUNK")) {   // tuning hook: columns per chunk (0 = no pipelining)
        const long v = atol(e);
        cw = v <= 0 || (uint64_t)v >= h->W ? W : (uint32_t)v;
    } else if (!h->thr && !h->force_block) {
        const uint64_t per_col = h->L / h->Ts;
        if (per_col > 0) {
            uint64_t unit = (2ull * 148 * 14) / per_col;
            if (unit == 0) unit = 1;
            if (2 * unit <= W) cw = (uint32_t)unit;
        }
    }
    if (h->thr || h->force_block) cw = W;
    // chunk boundaries: a short first chunk (its copy is the only exposed one), then chunks that grow by the factor by
    // which copying a column is faster than sweeping it n_sweeps times, so that chunk c+1 has arrived when chunk c is
    // done while the later, larger launches lose less to launch and tail overhead; at most four times the first.  The
    // factor is an estimate from the measured configs (a sweep of a column costs about 0.0164 of its copy per Philox
    // block executed per attempt: cfg4 ~12 blocks, ten sweeps: 2.0; cfg3 ~6.4 blocks: 1.05), clamped to [1, 2].
    // PCPD_STEP_CHUNK: uniform chunks.
    uint32_t bounds[66];
    uint32_t nchunks = 0;
    bounds[0] = 0;
    {
        const uint32_t nbd = (h->P.thd.nplanes + 1u) >> 1, nbp = (h->P.thp.nplanes + 1u) >> 1;
        const double blocks = 1.0 + (nbd >= 5 ? 6.5 : nbd ? 1.0 : 0.0) + (h->P.pmask_paper ? 1.0 : nbp >= 5 ? 4.7 : nbp ? 1.0 : 0.0);
        double grow = 0.0164 * blocks * (double)n_sweeps;
        grow = grow < 1.0 ? 1.0 : grow > 2.0 ? 2.0 : grow;
        if (getenv("PCPD_STEP_CHUNK")) grow = 1.0;
        uint32_t w0 = 0;
        double mult = 1.0;   // chunk size in units of cw: whole multiples, so that every launch stays wave-aligned
        while (w0 < W && nchunks < 64) {
            const uint32_t sz = cw * (uint32_t)(mult + 0.5);
            const uint32_t nw = (W - w0 < sz + cw || nchunks == 63) ? W - w0 : sz;   // (a last chunk below one unit is merged)
            w0 += nw;
            bounds[++nchunks] = w0;
            if (mult * grow <= 4.0) mult *= grow;
        }
    }
    int rc = ensure_copy_resources(h, nchunks);
    if (rc != PCPD_OK) return rc;
    cudaStream_t copy = h->copy_stream;
    cudaEvent_t *ev = h->chunk_ev;
    h->invalid = true;   // the lattice is overwritten chunk by chunk (see pcpd_step_from_host)
    cudaError_t e = cudaEventRecord(h->copy_start, h->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(copy, h->copy_start, 0);
    for (uint32_t c = 0; e == cudaSuccess && c < nchunks; ++c) {
        const uint32_t w0 = bounds[c], nw = bounds[c + 1] - w0;
        e = cudaMemcpyAsync(h->lat + (size_t)w0 * L, in_columns + (size_t)w0 * L, (size_t)nw * L * 8, cudaMemcpyHostToDevice, copy);
        if (e == cudaSuccess) e = cudaEventRecord(ev[c], copy);
    }
    for (uint32_t c = 0; e == cudaSuccess && c < nchunks; ++c) {
        const uint32_t w0 = bounds[c], nw = bounds[c + 1] - w0;
        e = cudaStreamWaitEvent(h->stream, ev[c], 0);
        if (e != cudaSuccess) break;
        SweepParams Pc = h->P;   // the chunk as a lattice of its own: columns w0 .. w0+nw-1 (columns never interact)
        Pc.lat = h->lat + (size_t)w0 * L;
        Pc.W = nw;
        Pc.word_offset = h->P.word_offset + w0;
        if (h->thr) Pc.thr_dev = h->thr + 4 * (size_t)w0;
        for (uint64_t it = 0; it < n_sweeps; ++it) {
            Pc.t = (uint32_t)(h->sweep + it);
            g_launches += launch_sweep(Pc, h->variant, h->force_block, h->stream, &h->jit, nchunks == 1 ? &h->split : nullptr);
        }
    }
    if (e == cudaSuccess) rc = check_launch("pipelined step");
    if (e == cudaSuccess && rc == PCPD_OK) {
        h->sweep += n_sweeps;
        h->invalid = false;
        if (out_counts) rc = pcpd_density(h, out_counts);
        else e = cudaStreamSynchronize(h->stream);
    }
    cudaStreamSynchronize(copy);
    cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(e, "step_from_host_columns");
    return rc;
}

int pcpd_step_from_host(pcpd_t *h, const uint64_t *in_words, uint64_t n_sweeps, uint32_t *out_counts)
{
    if (!h || !in_words) return fail(PCPD_ERR_ARG, "null argument");
    if (h->sweep + n_sweeps > 0xffffffffull) return fail(PCPD_ERR_RANGE, "sweep counter would exceed 2^32-1");
    const uint32_t cw = step_chunk_columns(h);
    const uint32_t L = (uint32_t)h->L, W = (uint32_t)h->W;
    if (cw >= W || h->thr || h->force_block) {   // no pipelining: the plain sequence
        int rc = pcpd_set_lattice(h, in_words);
        if (rc == PCPD_OK) rc = pcpd_run(h, n_sweeps);
        if (rc == PCPD_OK && out_counts) rc = pcpd_density(h, out_counts);
        return rc;
    }
    const size_t bytes = 8 * h->L * h->W;
    const uint32_t nchunks = (W + cw - 1) / cw;
    int rc0 = ensure_copy_resources(h, nchunks);
    if (rc0 != PCPD_OK) return rc0;
    cudaError_t e = cudaSuccess;
    uint64_t *stage = (uint64_t *)dev_alloc(h->mem, bytes, h->stream);
    if (!stage) return fail(PCPD_ERR_ALLOC, "staging allocation failed");
    cudaStream_t copy = h->copy_stream;
    cudaEvent_t *ev = h->chunk_ev;
    // From here on the lattice is overwritten chunk by chunk: a failure leaves it partly new, partly swept, so the
    // handle is marked invalid until the whole step has been queued without error (pcpd.h).
    h->invalid = true;
    // the copies start once everything already queued on the handle's stream has finished with the lattice
    e = cudaEventRecord(h->copy_start, h->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(copy, h->copy_start, 0);
    for (uint32_t c = 0; e == cudaSuccess && c < nchunks; ++c) {
        const uint32_t w0 = c * cw, nw = (w0 + cw <= W ? cw : W - w0);
        uint64_t *dst = stage + (size_t)w0 * L;   // chunk held densely as [L][nw]
        e = cudaMemcpy2DAsync(dst, (size_t)nw * 8, in_words + w0, (size_t)W * 8, (size_t)nw * 8, L, cudaMemcpyHostToDevice, copy);
        if (e == cudaSuccess) e = cudaEventRecord(ev[c], copy);
    }
    int rc = PCPD_OK;
    for (uint32_t c = 0; e == cudaSuccess && rc == PCPD_OK && c < nchunks; ++c) {
        const uint32_t w0 = c * cw, nw = (w0 + cw <= W ? cw : W - w0);
        e = cudaStreamWaitEvent(h->stream, ev[c], 0);
        if (e != cudaSuccess) break;
        g_launches += launch_transpose(stage + (size_t)w0 * L, h->lat + (size_t)w0 * L, L, nw, 1, h->stream);
        SweepParams Pc = h->P;   // the chunk as a lattice of its own: columns w0 .. w0+nw-1 (columns never interact)
        Pc.lat = h->lat + (size_t)w0 * L;
        Pc.W = nw;
        Pc.word_offset = h->P.word_offset + w0;
        for (uint64_t it = 0; it < n_sweeps; ++it) {
            Pc.t = (uint32_t)(h->sweep + it);
            g_launches += launch_sweep(Pc, h->variant, false, h->stream, &h->jit, nullptr);
        }
    }
    if (e == cudaSuccess && rc == PCPD_OK) rc = check_launch("pipelined step");
    if (e == cudaSuccess && rc == PCPD_OK) {
        h->sweep += n_sweeps;
        h->invalid = false;
        if (out_counts) rc = pcpd_density(h, out_counts);
        else e = cudaStreamSynchronize(h->stream);
    }
    cudaStreamSynchronize(copy);
    cudaStreamSynchronize(h->stream);
    dev_free(h->mem, stage);
    if (e != cudaSuccess) return cuda_fail(e, "step_from_host");
    return rc;
}

int pcpd_schedule_info(const pcpd_t *h, uint32_t *Ts, uint32_t *D, uint32_t *A, uint32_t *K)
{
    if (!h) return fail(PCPD_ERR_ARG, "null handle");
    if (Ts) *Ts = h->Ts;
    if (D) *D = h->D;
    if (A) *A = h->A;
    if (K) *K = 32;
    return PCPD_OK;
}

int pcpd_thresholds(const pcpd_t *h, uint64_t *Td, uint64_t *Tp)
{
    if (!h) return fail(PCPD_ERR_ARG, "null handle");
    if (Td) *Td = h->Td;
    if (Tp) *Tp = h->Tp;
    return PCPD_OK;
}

uint64_t pcpd_sweep(const pcpd_t *h) { return h ? h->sweep : 0; }

int pcpd_set_sweep(pcpd_t *h, uint64_t sweep)
{
    if (!h) return fail(PCPD_ERR_ARG, "null handle");
    if (sweep > 0xffffffffull) return fail(PCPD_ERR_RANGE, "sweep counter must be < 2^32");
    h->sweep = sweep;
    return PCPD_OK;
}

int pcpd_synchronize(pcpd_t *h)
{
    if (!h) return fail(PCPD_ERR_ARG, "null handle");
    const cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(e, "synchronize");
    return PCPD_OK;
}

int pcpd_jit_state(const pcpd_t *h) { return h ? h->jit.state : 0; }
uint64_t pcpd_split_launch_count(const pcpd_t *h) { return h ? h->split.launches : 0; }
const char *pcpd_jit_message(void) { return jit_message(); }
uint64_t pcpd_jit_launch_count(void) { return jit_launch_count(); }

int pcpd_jit_selftest(int variant, uint32_t T_d, uint32_t T_p, uint64_t *cubin_bytes)
{
    if (variant < 0 || variant > 3) return fail(PCPD_ERR_ARG, "jit_selftest: unknown variant %d", variant);
    size_t n = 0;
    JitSpec js;
    js.variant = variant; js.wpb = 7; js.pmode = 0;
    js.nud = T_d ? (int)((32 - __builtin_ctz(T_d) + 1) / 2 < 6 ? (32 - __builtin_ctz(T_d) + 1) / 2 : 6) : 0;
    js.nup = T_p ? (int)((32 - __builtin_ctz(T_p) + 1) / 2 < 4 ? (32 - __builtin_ctz(T_p) + 1) / 2 : 4) : 0;
    js.Td = T_d; js.Tp = T_p; js.Ts = PCPD_DEFAULT_TS; js.D = PCPD_DEFAULT_D; js.A = PCPD_DEFAULT_A; js.L = 1u << 20;
    if (jit_compile_only(js, &n) != 0) return fail(PCPD_ERR_DEVICE, "%s", jit_message());
    if (cubin_bytes) *cubin_bytes = n;
    return PCPD_OK;
}

int pcpd_microbench(int kind, uint32_t iters, double *out_rate)
{
    if (kind < 0 || kind >= microbench_kinds() || !out_rate || iters == 0) return fail(PCPD_ERR_ARG, "microbench: bad arguments");
    const int rc = run_microbench(kind, iters, out_rate, nullptr);
    g_launches += 4;
    if (rc != 0) return fail(rc, "microbench failed");
    return check_launch("microbench kernel");
}

}  // extern "C"
