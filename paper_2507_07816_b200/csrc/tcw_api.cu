// tcw_api.cu -- host runtime and C ABI of libtcw.so (declared in include/tcw.h).
//
// The host side validates arguments, owns the device copies (spectrogram re-laid to a 16-byte
// aligned pitch with PAD_BINS zero bins on both sides of every row, bit-packed counts expanded
// to one byte per bin; timestamps; velocities), the grow-only scratch (tables, grid axes,
// per-tile candidates) and the launch plan.  Every step of the path runs in the kernels of
// tcw_tables.cuh and tcw_sum.cuh; there is no CPU fallback.
#include "../../include/tcw.h"

#include <cuda.h>           // driver API types only (cuStreamWaitValue32 is fetched at run time; no link dependency)
#include <cuda_runtime.h>
#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "tcw_sum.cuh"
#include "tcw_tables.cuh"
#include "tcw_skyblock.cuh"
#include "tcw_skyblock2.cuh"
#include "tcw_bank.cuh"
#include "tcw_select.cuh"
#include "tcw_prep.cuh"
#include "tcw_peaks.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(call)                                                                         \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(e_ == cudaErrorMemoryAllocation ? TCW_ENOMEM : TCW_ECUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                               \
    } while (0)

constexpr double C_LIGHT = 299792458.0;
constexpr size_t SMEM_MAX = 227 * 1024;
constexpr long TOPK_TWO_READ_MIN = 1L << 22;   // tcw_topk: arrays of at least this many values take the two-read route
constexpr size_t TIMING_MAX = 4096;  // timed searches kept between two tcw_get_timing calls
// staged kernel, SFT chunking: used when the spectrogram rows of the span exceed CHUNK_MIN_BYTES;
// a chunk then holds about CHUNK_TARGET_BYTES of rows (inside the 126 MB L2) and at most
// CHUNK_MAX_ROWS rows (measured on B200: cfg4 is fastest at 1024-1280 rows of 80 KB, cfg2 at 2048
// rows of 16 KB; chunk-size sweeps of round 1d)
constexpr double CHUNK_MIN_BYTES = 96e6, CHUNK_TARGET_BYTES = 80e6, CHUNK_SCRATCH_MAX = 16e9;
constexpr long CHUNK_MAX_ROWS = 2048;

// ---- device memory: a library-owned stream-ordered pool ---------------------------------------
// cudaMalloc / cudaFree cost tens to hundreds of microseconds each and synchronise the device; a
// create / search / destroy cycle makes about fifteen of them.  All device memory of the library
// therefore comes from one CUDA memory pool per device (cudaMallocFromPoolAsync / cudaFreeAsync on
// the call's stream) that keeps up to POOL_KEEP_BYTES of freed blocks for the next handle.  If the
// pool cannot be created the calls fall back to cudaMalloc / cudaFree.
constexpr unsigned long long POOL_KEEP_BYTES = 8ull << 30;
thread_local cudaStream_t g_alloc_stream = nullptr;   // stream of the API call in progress on this thread

cudaMemPool_t library_pool()
{
    static std::mutex mu;
    static cudaMemPool_t pools[64];
    static int state[64];   // 0 not tried, 1 ready, -1 unavailable
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (state[dev] == 0) {
        cudaMemPoolProps props;
        std::memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        unsigned long long keep = POOL_KEEP_BYTES;
        if (cudaMemPoolCreate(&pools[dev], &props) == cudaSuccess &&
            cudaMemPoolSetAttribute(pools[dev], cudaMemPoolAttrReleaseThreshold, &keep) == cudaSuccess)
            state[dev] = 1;
        else {
            state[dev] = -1;
            cudaGetLastError();
        }
    }
    return state[dev] == 1 ? pools[dev] : nullptr;
}

cudaError_t dev_alloc(void **p, size_t bytes, cudaStream_t st)
{
    cudaMemPool_t pool = library_pool();
    if (pool) return cudaMallocFromPoolAsync(p, std::max<size_t>(bytes, 1), pool, st);
    return cudaMalloc(p, std::max<size_t>(bytes, 1));
}

void dev_free(void *p, cudaStream_t st)
{
    if (!p) return;
    if (library_pool()) cudaFreeAsync(p, st);
    else cudaFree(p);
}

// Progress counters of the progressive read-back (tcw_search_host): stream memory operations
// (cuStreamWaitValue32) need a plain cudaMalloc allocation, not pool memory, and cudaMalloc / cudaFree per
// handle would cost more than the read-back saves.  One block of PROGRESS_SLOTS x 16 counters per device,
// allocated on first use and kept; handles borrow a slot.
constexpr int PROGRESS_SLOTS = 256;
struct ProgressPool {
    std::mutex mu;
    unsigned int *base[64] = {nullptr};
    std::vector<int> free_slots[64];
};
ProgressPool &progress_pool()
{
    static ProgressPool pool;
    return pool;
}
unsigned int *progress_acquire(int dev)
{
    if (dev < 0 || dev >= 64) return nullptr;
    ProgressPool &pp = progress_pool();
    std::lock_guard<std::mutex> lock(pp.mu);
    if (!pp.base[dev]) {
        if (cudaMalloc((void **)&pp.base[dev], (size_t)PROGRESS_SLOTS * 16 * sizeof(unsigned int)) != cudaSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        for (int i = PROGRESS_SLOTS - 1; i >= 0; --i) pp.free_slots[dev].push_back(i);
    }
    if (pp.free_slots[dev].empty()) return nullptr;
    const int slot = pp.free_slots[dev].back();
    pp.free_slots[dev].pop_back();
    return pp.base[dev] + 16 * slot;
}
void progress_release(int dev, unsigned int *p)
{
    if (!p || dev < 0 || dev >= 64) return;
    ProgressPool &pp = progress_pool();
    std::lock_guard<std::mutex> lock(pp.mu);
    pp.free_slots[dev].push_back((int)((p - pp.base[dev]) / 16));
}

// grow-only device buffer; allocates on the stream of the API call in progress
template <typename T> struct DevBuf {
    T *p = nullptr;
    size_t cap = 0;  // elements
    int reserve(size_t n)
    {
        if (n <= cap) return TCW_OK;
        if (p) {
            cudaDeviceSynchronize();   // rare (a later search needs more scratch): nothing may still read the old block
            dev_free(p, g_alloc_stream);
        }
        p = nullptr;
        cap = 0;
        CUDA_TRY(dev_alloc((void **)&p, std::max<size_t>(n, 1) * sizeof(T), g_alloc_stream));
        cap = n;
        return TCW_OK;
    }
    void release()
    {
        dev_free(p, g_alloc_stream);
        p = nullptr;
        cap = 0;
    }
};

size_t row_bytes(int format, int n_bins)
{
    switch (format) {
    case TCW_F32_POWER: return 4 * (size_t)n_bins;
    case TCW_U8_COUNT: return (size_t)n_bins;
    default: return 4 * (((size_t)n_bins + 31) / 32);
    }
}

bool is_pow2(double x)
{
    int e;
    return x > 0 && std::isfinite(x) && std::frexp(x, &e) == 0.5;
}

// The library's copy of the spectrogram as a rank-3 tensor [n_sft][pitch/128][128 bytes] and, for n = 1 .. BOX_SEG_MAX,
// the map whose box is {128 bytes, n segments, RB rows}: the RB consecutive SFT rows of one ring slot of the staged kernel,
// n*128 bytes of each, in ONE TMA copy (cp.async.bulk.tensor.3d).  maps[0] is unused.  Out-of-range parts of a box read as
// zero.  cuTensorMapEncodeTiled is fetched at run time (no link dependency on libcuda).
constexpr int BOX_SEG_MAX = 31;
bool encode_box_maps(const void *base, long pitch, int n_sft, std::vector<CUtensorMap> &maps)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = [] {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            fn = nullptr;
        cudaGetLastError();
        return (encode_fn)fn;
    }();
    if (!encode || pitch % 128 != 0 || ((uintptr_t)base & 127) != 0) return false;
    maps.assign(BOX_SEG_MAX + 1, CUtensorMap());
    const cuuint64_t dims[3] = {128, (cuuint64_t)(pitch / 128), (cuuint64_t)n_sft};
    const cuuint64_t strides[2] = {128, (cuuint64_t)pitch};
    const cuuint32_t es[3] = {1, 1, 1};
    for (int n = 1; n <= BOX_SEG_MAX; ++n) {
        const cuuint32_t box[3] = {128, (cuuint32_t)n, (cuuint32_t)tcw::RB};
        if (encode(&maps[n], CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void *>(base), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    return true;
}

}  // namespace

struct tcw_handle {
    int device = 0;
    int format = 0, n_sft = 0, n_bins = 0, k_min = 0;
    int fmt_dev = 0;   // device format of the library's copy: tcw::FMT_F32 or tcw::FMT_U8
    long pitch = 0;    // its row pitch in bytes, padding included
    long pad_bytes = 0;
    double f_min = 0, T = 0;
    bool t_pow2 = false;
    double vmax = 0;  // max |v_j|
    int count_max = 1;  // count formats: largest element of the spectrogram (1 for bit-packed input)
    bool count_known = true;  // false while an asynchronous uint8 upload has not been scanned yet
    double vmid[3] = {0, 0, 0};  // velocity at the middle SFT: sort key of the sky-block kernel
    std::vector<double> ts;
    unsigned char *d_spec = nullptr;
    unsigned char *d_tmaps = nullptr;  // staged kernel: CUtensorMap n at d_tmaps + 128*n, box {128 bytes, n segments, RB rows}
    int max_seg = 0;                   // ... for n = 1 .. max_seg (0: no tensor maps, 1-D bulk copies only)
    double *d_ts = nullptr, *d_vel = nullptr;
    // grow-only scratch
    DevBuf<double> d_g, d_d, d_axes;
    DevBuf<unsigned char> d_partial, d_stat, d_best;
    DevBuf<unsigned char> d_cpart, d_clive;  // chunked staged searches: per-chunk partial sums, live flags
    DevBuf<unsigned char> d_selws;           // selection scratch (histogram, state, block counts, candidates)
    DevBuf<unsigned char> d_selzoom;         // top-K two-read route: per-CTA histograms, candidate keys and indices
    DevBuf<double> d_bank;                   // bank searches: f0, tau, brk [n] and sky [n][3] or [3]
    unsigned long long *d_counter = nullptr; // bank searches: lookups decided by the defining chain
    DevBuf<float> d_w;                       // weighted searches: weights [n_sky][n_sft]
    DevBuf<double> d_cw;                     // weighted searches: per-chunk sums of w and w^2 (float64)
    DevBuf<long> d_sel;
    DevBuf<double> d_dts, d_dmm;  // sky-block kernel: per-block Doppler rows and their {min, max}
    DevBuf<int> d_slot;           // sky index of each block slot
    std::vector<int> slot_host;
    int *d_status = nullptr;
    double *h_stage = nullptr;  // pinned staging for the grid axes / selections
    size_t h_stage_cap = 0;     // bytes
    cudaEvent_t ev_stage = nullptr;
    // options
    int opt_kernel = 0, opt_timing = 0, opt_r = 0, opt_stages = 0, opt_sky = 0, opt_exact = 0;
    long opt_chunk = 0;  // SFT rows per chunk of the staged kernel: 0 auto, -1 never chunk
    cudaStream_t dl_stream = nullptr;        // tcw_search_host: read-back stream
    cudaEvent_t dl_ready = nullptr;          // recorded once the progress counters of a search have been cleared
    unsigned int *d_progress = nullptr;      // per-part completion counters of a progressive search (a borrowed slot
                                             // of the library's cudaMalloc block: see progress_acquire)
    int want_parts = 0;                      // set by tcw_search_host: cut the (tau, n) axis into this many parts
    bool progress_active = false;            // the last search_impl ran with progress counters
    int progress_np = 0;                     // ... over this many parts
    unsigned int progress_target[16] = {0};  // CTAs per part
    int progress_a0[17] = {0};               // tau index where each part starts
    int opt_nonuniform = 0;   // 1: never take the equally-spaced-f0 instantiation of the staged kernel
    int opt_row_copies = 0;   // 1: never stage a ring slot by one tensor-map copy
    long plan_groups = 0;     // tcw_search_groups: group count of the WHOLE grid while its sub-grids are searched (chunk plan)
    double chunk_scratch_max = CHUNK_SCRATCH_MAX;   // lowered by the test hook TCW_OPT_DEBUG_CHUNK_SCRATCH
    bool keep_status = false; // a multi-part search (tcw_search_groups, tcw_search_host) clears the status word once
    int dbg_slot_shrink = 0;  // test hook: bytes taken off the kernels' own window bound
    int dbg_fail_wait = 0;    // test hook: the stream wait of read-back part (value - 1) reports CUDA_ERROR_NOT_SUPPORTED
    std::vector<cudaEvent_t> ev;  // 4 per timed search: start, tables done, sum done, best done
    size_t timing_n = 0;          // timed searches recorded since the last tcw_get_timing
    cudaStream_t last_stream = nullptr;
    // asynchronous upload (tcw_create_async): pieces of rows copied on up_stream, one event per piece
    cudaStream_t up_stream = nullptr;
    std::vector<cudaEvent_t> up_ev;
    std::vector<long> up_end;    // one past the last row of each piece
    bool up_pending = false;     // the first search still has to wait for the pieces
    void *up_staging = nullptr;  // tightly packed device copy the pieces land in before the re-lay
    long info[12] = {0, 0, 0, 0, 0, 0, 0, 0, 1, 0, 0, 0};
    // last tables
    int tab_tau = 0, tab_brk = 0, tab_sky = 0;
    // device axis pointers of the last prepared grid
    const double *a_f0 = nullptr, *a_tau = nullptr, *a_brk = nullptr, *a_sky = nullptr;
};

namespace {

// The kernels set the device status word when a window bound computed on the host is violated
// (rows are then skipped, so the sums would be wrong).  Call with the search's stream synchronised.
int check_status(tcw_handle *h)
{
    int status = 0;
    CUDA_TRY(cudaMemcpy(&status, h->d_status, sizeof(int), cudaMemcpyDeviceToHost));
    h->info[4] = status;
    if (status != 0)
        return fail(TCW_EINTERNAL, "device status word %d: a staged window exceeded the bound planned on the host; "
                                   "the results of the last search on this handle are not valid", status);
    return TCW_OK;
}

// Start of an API call on `st`: scratch of this call is allocated on st; if the previous call on
// this handle used another stream, wait for it (buffers are reused across calls).
void enter(tcw_handle *h, cudaStream_t st)
{
    if (h->last_stream != st) cudaStreamSynchronize(h->last_stream);
    g_alloc_stream = st;
}

int validate_grid(const tcw_handle *h, const tcw_grid *g)
{
    if (!g) return fail(TCW_EINVAL, "grid is NULL");
    if (g->n_f0 <= 0 || g->n_tau <= 0 || g->n_brk <= 0 || g->n_sky <= 0)
        return fail(TCW_EINVAL, "grid sizes must be positive");
    if (!g->f0 || !g->tau || !g->brk || !g->sky) return fail(TCW_EINVAL, "grid axis pointer is NULL");
    if (!std::isfinite(g->T0)) return fail(TCW_EINVAL, "T0 is not finite");
    for (int i = 0; i < g->n_f0; ++i) {
        if (!(g->f0[i] > 0) || !std::isfinite(g->f0[i])) return fail(TCW_EINVAL, "f0[%d] must be > 0", i);
        if (i && !(g->f0[i] > g->f0[i - 1])) return fail(TCW_EINVAL, "f0 must be strictly ascending (at %d)", i);
    }
    if (g->f0[g->n_f0 - 1] * h->T >= 2147483648.0 - 1048576.0)
        return fail(TCW_EINVAL, "f0_max*T_sft exceeds the 32-bit bin range");
    for (int i = 0; i < g->n_tau; ++i)
        if (!(g->tau[i] > 0) || !std::isfinite(g->tau[i])) return fail(TCW_EINVAL, "tau[%d] must be > 0", i);
    for (int i = 0; i < g->n_brk; ++i)
        if (!(g->brk[i] > 1) || !std::isfinite(g->brk[i])) return fail(TCW_EINVAL, "braking index brk[%d] must be > 1", i);
    for (int i = 0; i < g->n_sky; ++i) {
        const double *n = g->sky + 3 * (size_t)i;
        double nrm = std::sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        if (!(std::fabs(nrm - 1.0) <= 1e-6)) return fail(TCW_EINVAL, "sky[%d] is not a unit vector", i);
    }
    long n_groups = 0, n_templates = 0;
    if (__builtin_mul_overflow((long)g->n_sky, (long)g->n_tau, &n_groups) ||
        __builtin_mul_overflow(n_groups, (long)g->n_brk, &n_groups) ||
        __builtin_mul_overflow(n_groups, (long)g->n_f0, &n_templates) || n_groups > (1L << 40) ||
        n_templates > (1L << 48))
        return fail(TCW_EINVAL, "grid too large");
    return TCW_OK;
}

int ensure_stage(tcw_handle *h, size_t bytes)
{
    if (bytes <= h->h_stage_cap) return TCW_OK;
    if (h->h_stage) cudaFreeHost(h->h_stage);
    h->h_stage = nullptr;
    h->h_stage_cap = 0;
    CUDA_TRY(cudaMallocHost((void **)&h->h_stage, bytes));
    h->h_stage_cap = bytes;
    return TCW_OK;
}

// Copy the grid axes (and an optional selection list) to the device through pinned staging,
// then build both tables on `st`.
int prepare(tcw_handle *h, const tcw_grid *g, long n_sel, const long *sel, cudaStream_t st,
            const std::vector<int> *slots = nullptr)
{
    CUDA_TRY(cudaSetDevice(h->device));
    const size_t n_axes = (size_t)g->n_f0 + g->n_tau + g->n_brk + 3 * (size_t)g->n_sky;
    const size_t n_slots = slots ? slots->size() : 0;
    const size_t stage_bytes = n_axes * sizeof(double) + (size_t)std::max<long>(n_sel, 0) * sizeof(long) +
                               n_slots * sizeof(int);
    // the staging buffer may still feed the previous call's copy
    CUDA_TRY(cudaEventSynchronize(h->ev_stage));
    int rc;
    if ((rc = ensure_stage(h, stage_bytes)) != TCW_OK) return rc;
    if ((rc = h->d_axes.reserve(n_axes)) != TCW_OK) return rc;
    if ((rc = h->d_g.reserve((size_t)g->n_tau * g->n_brk * h->n_sft)) != TCW_OK) return rc;
    if ((rc = h->d_d.reserve((size_t)g->n_sky * h->n_sft)) != TCW_OK) return rc;
    if (n_sel > 0 && (rc = h->d_sel.reserve((size_t)n_sel)) != TCW_OK) return rc;
    if (n_slots && (rc = h->d_slot.reserve(n_slots)) != TCW_OK) return rc;

    double *w = h->h_stage;
    std::memcpy(w, g->f0, sizeof(double) * g->n_f0);
    std::memcpy(w + g->n_f0, g->tau, sizeof(double) * g->n_tau);
    std::memcpy(w + g->n_f0 + g->n_tau, g->brk, sizeof(double) * g->n_brk);
    std::memcpy(w + g->n_f0 + g->n_tau + g->n_brk, g->sky, sizeof(double) * 3 * (size_t)g->n_sky);
    CUDA_TRY(cudaMemcpyAsync(h->d_axes.p, w, n_axes * sizeof(double), cudaMemcpyHostToDevice, st));
    if (n_sel > 0) {
        std::memcpy(w + n_axes, sel, sizeof(long) * (size_t)n_sel);
        CUDA_TRY(cudaMemcpyAsync(h->d_sel.p, w + n_axes, sizeof(long) * (size_t)n_sel, cudaMemcpyHostToDevice, st));
    }
    if (n_slots) {
        int *ws = (int *)((char *)w + n_axes * sizeof(double) + (size_t)std::max<long>(n_sel, 0) * sizeof(long));
        std::memcpy(ws, slots->data(), n_slots * sizeof(int));
        CUDA_TRY(cudaMemcpyAsync(h->d_slot.p, ws, n_slots * sizeof(int), cudaMemcpyHostToDevice, st));
    }
    CUDA_TRY(cudaEventRecord(h->ev_stage, st));
    h->a_f0 = h->d_axes.p;
    h->a_tau = h->a_f0 + g->n_f0;
    h->a_brk = h->a_tau + g->n_tau;
    h->a_sky = h->a_brk + g->n_brk;

    if ((long)g->n_sky * h->n_sft > (1L << 38) || (long)g->n_tau * h->n_sft > (1L << 37))
        return fail(TCW_EUNSUPPORTED, "table of %ld x %d entries needs more than 2^31-1 CTAs; split the search", (long)g->n_sky, h->n_sft);
    {
        long total = (long)g->n_sky * h->n_sft;
        tcw::doppler_table_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(h->d_vel, h->n_sft, h->a_sky,
                                                                                 g->n_sky, h->d_d.p);
        CUDA_TRY(cudaGetLastError());
    }
    {
        long total = (long)g->n_tau * h->n_sft;
        tcw::spindown_table_kernel<<<(unsigned)((total + 127) / 128), 128, 0, st>>>(
            h->d_ts, h->n_sft, g->T0, h->a_tau, g->n_tau, h->a_brk, g->n_brk, h->d_g.p);
        CUDA_TRY(cudaGetLastError());
    }
    h->tab_tau = g->n_tau;
    h->tab_brk = g->n_brk;
    h->tab_sky = g->n_sky;
    h->last_stream = st;
    return TCW_OK;
}

tcw::SumParams base_params(const tcw_handle *h, const tcw_grid *g)
{
    tcw::SumParams p;
    std::memset(&p, 0, sizeof p);
    p.spec = h->d_spec + h->pad_bytes;
    p.spec_pad = h->d_spec;
    p.pad_bytes = h->pad_bytes;
    p.pitch = h->pitch;
    p.tmaps = h->d_tmaps;
    p.max_seg = h->max_seg;
    p.n_sft = h->n_sft;
    p.n_bins = h->n_bins;
    p.k_min = h->k_min;
    p.T = h->T;
    p.gtab = h->d_g.p;
    p.dtab = h->d_d.p;
    p.f0 = h->a_f0;
    p.n_f0 = g->n_f0;
    p.n_ab = g->n_tau * g->n_brk;
    p.n_groups = (long)g->n_sky * g->n_tau * g->n_brk;
    p.chunk_rows = h->n_sft;
    p.n_chunks = 1;
    p.j_begin = (int)(std::lower_bound(h->ts.begin(), h->ts.end(), g->T0) - h->ts.begin());
    // |beta| <= |v| |n-hat| / c with | |n-hat| - 1 | <= 1e-6; a relative 1e-5 on beta is ample
    const double dmax = 1.0 + (h->vmax / C_LIGHT) * (1.0 + 1e-5) + 1e-15;
    p.dmaxT = dmax * h->T * (1.0 + 1e-12);
    p.status = h->d_status;
    // fast bin index of the staged kernel: |fast x - oracle's x| <= 3*x*2^-52 + 2^-32 bins;
    // thr is that bound with a margin, in units of 2^-32 bin, never below 64 units (1.5e-8 bin)
    {
        const double x_max = g->f0[g->n_f0 - 1] * p.dmaxT;
        const double units = std::ceil((4.0 * x_max * 0x1p-52 + 0x1p-31) * 0x1p32);
        double thr_units = std::max(64.0, units);
        // equally spaced f0 (the cubic lattice of PAPER.md:63): f0[i] = f0[0] + i*delta up to a deviation worth
        // less than 2^-34 bin.  The kernel then needs no per-template f0 registers.
        p.d32 = 0.0;
        if (g->n_f0 >= 2 && !h->opt_nonuniform) {
            // delta as the kernel will use it (a binary64 number); the deviation of the axis from f0[0] + i*delta is
            // measured in extended precision and, times the largest D*T, must stay below 2^-34 bin.  The kernel's own
            // roundings of lane*delta and 32*delta*c are relative 2^-53 errors on less than a window: far below that.
            const double d = (double)(((long double)g->f0[g->n_f0 - 1] - (long double)g->f0[0]) / (long double)(g->n_f0 - 1));
            long double dev = 0;
            for (int i = 0; i < g->n_f0; ++i)
                dev = std::max(dev, fabsl((long double)g->f0[i] - ((long double)g->f0[0] + (long double)i * (long double)d)));
            if (d > 0 && (double)dev * p.dmaxT <= 0x1p-34) {
                p.d32 = 32.0 * d;
                thr_units += 2.0;
            }
        }
        if (h->opt_exact || thr_units > 1048576.0) {
            p.thr2 = 0xffffffffu;
            p.fix_add = 0.5;
        } else {
            p.thr2 = (uint32_t)(2.0 * thr_units);
            p.fix_add = 0.5 + thr_units * 0x1p-32;
        }
    }
    return p;
}

// Upper bound of the number of bins a tile of `tile` consecutive f0 can select in one SFT:
// k_last - k_first + 1 <= (f_last - f_first) * T * g * D + 2 with g <= 1, D*T <= dmaxT.
long max_window_bins(const tcw_grid *g, int tile, double dmaxT)
{
    double df = 0;
    for (int i0 = 0; i0 < g->n_f0; i0 += tile) {
        int i1 = std::min(i0 + tile, g->n_f0) - 1;
        df = std::max(df, g->f0[i1] - g->f0[i0]);
    }
    // rint(x2) - rint(x1) <= floor(x2 - x1) + 1 for exact x; the relative 1e-9 covers the float64 error of the tracks
    double w = std::floor(df * dmaxT * (1.0 + 1e-9) + 1e-6) + 2.0;
    return w > 1e9 ? (long)1e9 : (long)w;
}

// Bytes of one staged row of a ring slot.  box = false: the window's bins plus the 16-byte alignment slack at both
// ends (a 1-D bulk copy per row).  box = true: a whole number of 128-byte segments that holds the window wherever it
// starts inside its first segment (one tensor-map copy per slot; the 1-D layout fits as well).
int slot_bytes_for(int fmt_dev, long w_bins, bool box)
{
    const long wb = fmt_dev == tcw::FMT_F32 ? 4 * w_bins : w_bins;
    long b = box ? (wb + 124 + 127) & ~127L : (wb + 32 + 15) & ~15L;
    return b > (1L << 30) ? (1 << 30) : (int)b;
}

template <int FMT, int R, bool P2, bool WGT, bool UNI>
int launch_staged_t(const tcw::SumParams &p, long n_ctas, size_t smem, cudaStream_t st)
{
    auto kern = tcw::sum_staged_kernel<FMT, R, P2, WGT, UNI>;
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)n_ctas, tcw::STAGED_THREADS, smem, st>>>(p);
    CUDA_TRY(cudaGetLastError());
    return TCW_OK;
}

template <int FMT, bool P2, bool WGT, bool UNI>
int launch_staged_r(int r, const tcw::SumParams &p, long n_ctas, size_t smem, cudaStream_t st)
{
    switch (r) {
    case 16: return launch_staged_t<FMT, 16, P2, WGT, UNI>(p, n_ctas, smem, st);
    case 8: return launch_staged_t<FMT, 8, P2, WGT, UNI>(p, n_ctas, smem, st);
    default: return launch_staged_t<FMT, 4, P2, WGT, UNI>(p, n_ctas, smem, st);
    }
}

template <bool WGT, bool UNI>
int launch_staged_w(int fmt, int r, bool p2, const tcw::SumParams &p, long n_ctas, size_t smem, cudaStream_t st)
{
    if (fmt == tcw::FMT_F32)
        return p2 ? launch_staged_r<tcw::FMT_F32, true, WGT, UNI>(r, p, n_ctas, smem, st)
                  : launch_staged_r<tcw::FMT_F32, false, WGT, UNI>(r, p, n_ctas, smem, st);
    return p2 ? launch_staged_r<tcw::FMT_U8, true, WGT, UNI>(r, p, n_ctas, smem, st)
              : launch_staged_r<tcw::FMT_U8, false, WGT, UNI>(r, p, n_ctas, smem, st);
}

// p.d32 != 0 selects the instantiation for an equally spaced f0 axis
int launch_staged(int fmt, int r, bool p2, bool wgt, const tcw::SumParams &p, long n_ctas, size_t smem, cudaStream_t st)
{
    if (p.d32 != 0.0)
        return wgt ? launch_staged_w<true, true>(fmt, r, p2, p, n_ctas, smem, st)
                   : launch_staged_w<false, true>(fmt, r, p2, p, n_ctas, smem, st);
    return wgt ? launch_staged_w<true, false>(fmt, r, p2, p, n_ctas, smem, st)
               : launch_staged_w<false, false>(fmt, r, p2, p, n_ctas, smem, st);
}

template <int FMT, bool WGT> int launch_gather_t(bool p2, const tcw::SumParams &p, long n_ctas, cudaStream_t st)
{
    if (p2) tcw::sum_gather_kernel<FMT, true, WGT><<<(unsigned)n_ctas, 128, 0, st>>>(p);
    else tcw::sum_gather_kernel<FMT, false, WGT><<<(unsigned)n_ctas, 128, 0, st>>>(p);
    CUDA_TRY(cudaGetLastError());
    return TCW_OK;
}

int launch_gather(int fmt, bool p2, bool wgt, const tcw::SumParams &p, long n_ctas, cudaStream_t st)
{
    if (wgt)
        return fmt == tcw::FMT_F32 ? launch_gather_t<tcw::FMT_F32, true>(p2, p, n_ctas, st)
                                   : launch_gather_t<tcw::FMT_U8, true>(p2, p, n_ctas, st);
    return fmt == tcw::FMT_F32 ? launch_gather_t<tcw::FMT_F32, false>(p2, p, n_ctas, st)
                               : launch_gather_t<tcw::FMT_U8, false>(p2, p, n_ctas, st);
}

template <int R, int SC, bool P2>
int launch_sky_t(const tcw::SumParams &p, const tcw::SkyParams &q, long n_ctas, size_t smem, cudaStream_t st)
{
    auto kern = tcw::sum_skyblock_kernel<R, SC, P2>;
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)n_ctas, tcw::SKY_THREADS, smem, st>>>(p, q);
    CUDA_TRY(cudaGetLastError());
    return TCW_OK;
}

int launch_sky(int sc, bool p2, const tcw::SumParams &p, const tcw::SkyParams &q, long n_ctas, size_t smem,
               cudaStream_t st)
{
    if (sc == 2) return p2 ? launch_sky_t<16, 2, true>(p, q, n_ctas, smem, st) : launch_sky_t<16, 2, false>(p, q, n_ctas, smem, st);
    return p2 ? launch_sky_t<8, 4, true>(p, q, n_ctas, smem, st) : launch_sky_t<8, 4, false>(p, q, n_ctas, smem, st);
}

int launch_sky_table(int sc, bool p2, const tcw_handle *h, const double *sky, int n_blocks, cudaStream_t st)
{
    const long warps = (long)n_blocks * h->n_sft;
    const unsigned blocks = (unsigned)((warps * 32 + 255) / 256);
#define TCW_SKY_TABLE(SC, P2)                                                                              \
    tcw::skyblock_table_kernel<SC, P2><<<blocks, 256, 0, st>>>(h->d_vel, h->n_sft, sky, h->d_slot.p, n_blocks, \
                                                               h->T, h->d_dts.p, h->d_dmm.p)
    if (sc == 2) { if (p2) TCW_SKY_TABLE(2, true); else TCW_SKY_TABLE(2, false); }
    else { if (p2) TCW_SKY_TABLE(4, true); else TCW_SKY_TABLE(4, false); }
#undef TCW_SKY_TABLE
    CUDA_TRY(cudaGetLastError());
    return TCW_OK;
}

}  // namespace

// =============================================================================== C ABI
extern "C" {

const char *tcw_last_error(void) { return g_err; }

static int create_impl(tcw_handle **out, const void *spectrogram, int format, long row_pitch_bytes, int n_sft,
                       int n_bins, double f_min, double T_sft, const double *timestamps, const double *velocities,
                       void *stream, bool async_upload)
{
    if (!out) return fail(TCW_EINVAL, "out is NULL");
    *out = nullptr;
    if (!spectrogram || !timestamps || !velocities) return fail(TCW_EINVAL, "NULL input pointer");
    if (format != TCW_F32_POWER && format != TCW_U8_COUNT && format != TCW_BIT_COUNT)
        return fail(TCW_EINVAL, "unknown spectrogram format %d", format);
    if (n_sft <= 0 || n_bins <= 0) return fail(TCW_EINVAL, "n_sft and n_bins must be positive");
    if (row_pitch_bytes < (long)row_bytes(format, n_bins))
        return fail(TCW_EINVAL, "row_pitch_bytes %ld is smaller than one row (%zu bytes)", row_pitch_bytes,
                    row_bytes(format, n_bins));
    if (!(T_sft > 0) || !std::isfinite(T_sft) || !(f_min >= 0) || !std::isfinite(f_min))
        return fail(TCW_EINVAL, "f_min must be >= 0 and T_sft > 0");
    const double km = std::rint(f_min * T_sft);
    if (std::fabs(f_min * T_sft - km) > 1e-9) return fail(TCW_EINVAL, "f_min*T_sft must be an integer (bin-aligned band start)");
    if (km + n_bins >= 2147483648.0 - 1048576.0) return fail(TCW_EINVAL, "band exceeds the 32-bit bin range");
    double vmax = 0;
    for (int j = 0; j < n_sft; ++j) {
        if (!std::isfinite(timestamps[j])) return fail(TCW_EINVAL, "timestamps[%d] is not finite", j);
        if (j && !(timestamps[j] > timestamps[j - 1]))
            return fail(TCW_EINVAL, "timestamps must be strictly increasing (at %d)", j);
        const double *v = velocities + 3 * (size_t)j;
        double n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        if (!std::isfinite(n) || n >= 0.5 * C_LIGHT) return fail(TCW_EINVAL, "velocities[%d] is not a physical velocity", j);
        vmax = std::max(vmax, n);
    }

    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    tcw_handle *h = new (std::nothrow) tcw_handle;
    if (!h) return fail(TCW_ENOMEM, "out of host memory");
    h->device = dev;
    h->format = format;
    h->n_sft = n_sft;
    h->n_bins = n_bins;
    h->f_min = f_min;
    h->T = T_sft;
    h->t_pow2 = is_pow2(T_sft);
    h->k_min = (int)km;
    h->vmax = vmax;
    for (int c = 0; c < 3; ++c) h->vmid[c] = velocities[3 * (size_t)(n_sft / 2) + c];
    h->ts.assign(timestamps, timestamps + n_sft);
    h->fmt_dev = format == TCW_F32_POWER ? tcw::FMT_F32 : tcw::FMT_U8;
    const size_t bpb = h->fmt_dev == tcw::FMT_F32 ? 4 : 1;
    const size_t dev_row = bpb * (size_t)n_bins;           // bytes of one row in the device format
    h->pad_bytes = (long)(bpb * tcw::PAD_BINS);            // multiple of 16
    // a multiple of 128: the tensor maps of the staged kernel see a row as pitch/128 segments of 128 bytes
    h->pitch = (long)((2 * (size_t)h->pad_bytes + dev_row + 127) & ~(size_t)127);
    cudaStream_t st = (cudaStream_t)stream;
    g_alloc_stream = st;
    h->last_stream = st;
    void *d_words = nullptr;   // staging of the caller's rows (bit-packed words, or tightly packed host rows)

#define CREATE_TRY(call)                                                                       \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            int rc_ = fail(e_ == cudaErrorMemoryAllocation ? TCW_ENOMEM : TCW_ECUDA, "%s: %s", #call, \
                           cudaGetErrorString(e_));                                            \
            dev_free(d_words, st);                                                             \
            tcw_destroy(h);                                                                    \
            return rc_;                                                                        \
        }                                                                                      \
    } while (0)

    CREATE_TRY(dev_alloc((void **)&h->d_spec, (size_t)h->pitch * n_sft, st));
    CREATE_TRY(dev_alloc((void **)&h->d_ts, sizeof(double) * n_sft, st));
    CREATE_TRY(dev_alloc((void **)&h->d_vel, sizeof(double) * 3 * (size_t)n_sft, st));
    CREATE_TRY(dev_alloc((void **)&h->d_status, sizeof(int), st));
    CREATE_TRY(dev_alloc((void **)&h->d_counter, sizeof(unsigned long long), st));
    CREATE_TRY(cudaMemsetAsync(h->d_counter, 0, sizeof(unsigned long long), st));
    CREATE_TRY(cudaEventCreateWithFlags(&h->ev_stage, cudaEventDisableTiming));
    CREATE_TRY(cudaMemsetAsync(h->d_status, 0, sizeof(int), st));
    // the padding on either side of every row must read as zero (the payload is overwritten by the copies below)
    CREATE_TRY(cudaMemset2DAsync(h->d_spec, (size_t)h->pitch, 0, (size_t)h->pad_bytes, (size_t)n_sft, st));
    CREATE_TRY(cudaMemset2DAsync(h->d_spec + h->pad_bytes + dev_row, (size_t)h->pitch, 0,
                                 (size_t)h->pitch - (size_t)h->pad_bytes - dev_row, (size_t)n_sft, st));
    {
        // tensor maps of the staged kernel (SumParams::tmaps); without the driver entry point the kernel
        // falls back to one 1-D bulk copy per row
        std::vector<CUtensorMap> maps;
        if (encode_box_maps(h->d_spec, h->pitch, n_sft, maps)) {
            CREATE_TRY(dev_alloc((void **)&h->d_tmaps, maps.size() * sizeof(CUtensorMap), st));
            CREATE_TRY(cudaMemcpyAsync(h->d_tmaps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, st));
            CREATE_TRY(cudaStreamSynchronize(st));     // `maps` is pageable host memory
            h->max_seg = (int)maps.size() - 1;
        }
    }
    if (format == TCW_BIT_COUNT) {
        // bit-packed input: stage the words on the device, then expand to one byte per bin
        const size_t wrow = row_bytes(format, n_bins);
        CREATE_TRY(dev_alloc(&d_words, wrow * n_sft, st));
        // contiguous rows travel in one piece: a strided copy of 10 800 rows of 500 bytes from the host
        // costs about 4 ms on B200 against 0.2 ms for the same 5.4 MB in one transfer
        if ((size_t)row_pitch_bytes == wrow)
            CREATE_TRY(cudaMemcpyAsync(d_words, spectrogram, wrow * n_sft, cudaMemcpyDefault, st));
        else
            CREATE_TRY(cudaMemcpy2DAsync(d_words, wrow, spectrogram, (size_t)row_pitch_bytes, wrow, (size_t)n_sft,
                                         cudaMemcpyDefault, st));
        const long total = (long)n_sft * n_bins;
        const unsigned blocks = (unsigned)std::min<long>((total + 255) / 256, 148L * 16);
        tcw::expand_bits_kernel<<<blocks, 256, 0, st>>>((const uint32_t *)d_words, (long)(wrow / 4), n_sft, n_bins,
                                                        h->d_spec + h->pad_bytes, h->pitch);
        CREATE_TRY(cudaGetLastError());
    } else {
        // A strided host-to-device copy runs well below the link rate (measured on B200: 173 MB in
        // 4.8 ms against 3.1 ms for the same bytes in one piece), so host rows that are contiguous
        // go to the device in one copy and are spread to the padded pitch by a device-to-device copy.
        cudaPointerAttributes attr;
        const bool on_device = cudaPointerGetAttributes(&attr, spectrogram) == cudaSuccess &&
                               (attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged);
        cudaGetLastError();
        if (async_upload && !on_device && (size_t)row_pitch_bytes == dev_row) {
            // tcw_create_async: the rows travel in pieces of about 16 MB on a copy stream of the handle's
            // own, each piece followed by its re-lay and an event; the first search waits per SFT chunk.
            CREATE_TRY(dev_alloc(&h->up_staging, dev_row * n_sft, st));
            {
                // highest priority: the re-lay copies must not queue behind the search's CTAs
                int prio_lo = 0, prio_hi = 0;
                cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
                CREATE_TRY(cudaStreamCreateWithPriority(&h->up_stream, cudaStreamNonBlocking, prio_hi));
            }
            cudaEvent_t ready;
            CREATE_TRY(cudaEventCreateWithFlags(&ready, cudaEventDisableTiming));
            cudaEventRecord(ready, st);                       // allocations and the zero fill precede the pieces
            cudaStreamWaitEvent(h->up_stream, ready, 0);
            cudaEventDestroy(ready);
            // pieces of 16 MB while the first search is waiting to start, 64 MB afterwards (fewer calls and events)
            const long rows16 = std::max<long>(64, (long)((16 << 20) / dev_row));
            long up_rows = rows16;
            for (long j0 = 0; j0 < n_sft; j0 += up_rows) {
                up_rows = h->up_end.size() < 8 ? rows16 : 4 * rows16;
                const size_t nr = (size_t)std::min<long>(up_rows, n_sft - j0);
                unsigned char *stg = (unsigned char *)h->up_staging + (size_t)j0 * dev_row;
                CREATE_TRY(cudaMemcpyAsync(stg, (const unsigned char *)spectrogram + (size_t)j0 * dev_row, nr * dev_row,
                                           cudaMemcpyHostToDevice, h->up_stream));
                CREATE_TRY(cudaMemcpy2DAsync(h->d_spec + h->pad_bytes + (size_t)j0 * h->pitch, (size_t)h->pitch, stg, dev_row,
                                             dev_row, nr, cudaMemcpyDeviceToDevice, h->up_stream));
                cudaEvent_t e;
                CREATE_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                h->up_ev.push_back(e);
                h->up_end.push_back(j0 + (long)nr);
                CREATE_TRY(cudaEventRecord(e, h->up_stream));
            }
            h->up_pending = true;
        } else if (!on_device && (size_t)row_pitch_bytes == dev_row) {
            CREATE_TRY(dev_alloc(&d_words, dev_row * n_sft, st));
            CREATE_TRY(cudaMemcpyAsync(d_words, spectrogram, dev_row * n_sft, cudaMemcpyHostToDevice, st));
            CREATE_TRY(cudaMemcpy2DAsync(h->d_spec + h->pad_bytes, (size_t)h->pitch, d_words, dev_row, dev_row,
                                         (size_t)n_sft, cudaMemcpyDeviceToDevice, st));
        } else {
            CREATE_TRY(cudaMemcpy2DAsync(h->d_spec + h->pad_bytes, (size_t)h->pitch, spectrogram, (size_t)row_pitch_bytes,
                                         dev_row, (size_t)n_sft, cudaMemcpyDefault, st));
        }
    }
    if (format == TCW_U8_COUNT && !h->up_pending) {
        // the largest count decides whether the two-level sky-block kernel may serve this data
        // (d_status doubles as the result word; it is cleared again below)
        tcw::max_u8_kernel<<<148 * 8, 256, 0, st>>>(h->d_spec + h->pad_bytes, h->pitch, n_sft, n_bins, h->d_status);
        CREATE_TRY(cudaGetLastError());
        CREATE_TRY(cudaMemcpyAsync(&h->count_max, h->d_status, sizeof(int), cudaMemcpyDeviceToHost, st));
        CREATE_TRY(cudaMemsetAsync(h->d_status, 0, sizeof(int), st));
    } else if (format == TCW_U8_COUNT) {
        h->count_max = 255;   // asynchronous upload: the data are not here yet; the first search scans them
        h->count_known = false;
    }
    CREATE_TRY(cudaMemcpyAsync(h->d_ts, timestamps, sizeof(double) * n_sft, cudaMemcpyHostToDevice, st));
    CREATE_TRY(cudaMemcpyAsync(h->d_vel, velocities, sizeof(double) * 3 * (size_t)n_sft, cudaMemcpyHostToDevice, st));
    CREATE_TRY(cudaEventRecord(h->ev_stage, st));
    CREATE_TRY(cudaStreamSynchronize(st));
#undef CREATE_TRY
    dev_free(d_words, st);
    *out = h;
    return TCW_OK;
}

int tcw_create(tcw_handle **out, const void *spectrogram, int format, long row_pitch_bytes, int n_sft,
               int n_bins, double f_min, double T_sft, const double *timestamps, const double *velocities,
               void *stream)
{
    return create_impl(out, spectrogram, format, row_pitch_bytes, n_sft, n_bins, f_min, T_sft, timestamps, velocities,
                       stream, false);
}

int tcw_create_async(tcw_handle **out, const void *spectrogram, int format, long row_pitch_bytes, int n_sft,
                     int n_bins, double f_min, double T_sft, const double *timestamps, const double *velocities,
                     void *stream)
{
    return create_impl(out, spectrogram, format, row_pitch_bytes, n_sft, n_bins, f_min, T_sft, timestamps, velocities,
                       stream, true);
}

// Make `st` wait for the uploaded rows [0, j_end) of a handle created by tcw_create_async.
static void upload_wait_rows(tcw_handle *h, long j_end, cudaStream_t st)
{
    if (!h->up_pending || h->up_ev.empty()) return;
    long k = (long)(std::lower_bound(h->up_end.begin(), h->up_end.end(), std::max<long>(j_end, 1)) - h->up_end.begin());
    k = std::min<long>(k, (long)h->up_ev.size() - 1);
    cudaStreamWaitEvent(st, h->up_ev[(size_t)k], 0);
}

// Every piece has been waited for on `st`: later calls need no waits; the staging copy goes back to the pool.
static void upload_done(tcw_handle *h, cudaStream_t st)
{
    if (!h->up_pending) return;
    h->up_pending = false;
    dev_free(h->up_staging, st);
    h->up_staging = nullptr;
}

int tcw_upload_wait(tcw_handle *h)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    if (h->up_stream) CUDA_TRY(cudaStreamSynchronize(h->up_stream));
    return TCW_OK;
}

int tcw_destroy(tcw_handle *h)
{
    if (!h) return TCW_OK;
    cudaSetDevice(h->device);
    // nothing enqueued by this handle may still be running when its memory goes back to the pool
    cudaStreamSynchronize(h->last_stream);
    if (h->dl_stream) {
        cudaStreamSynchronize(h->dl_stream);
        if (h->dl_ready) cudaEventDestroy(h->dl_ready);
        cudaStreamDestroy(h->dl_stream);
    }
    if (h->up_stream) {
        cudaStreamSynchronize(h->up_stream);
        for (auto &e : h->up_ev) cudaEventDestroy(e);
        cudaStreamDestroy(h->up_stream);
    }
    g_alloc_stream = h->last_stream;
    dev_free(h->up_staging, h->last_stream);
    dev_free(h->d_spec, h->last_stream);
    dev_free(h->d_tmaps, h->last_stream);
    dev_free(h->d_ts, h->last_stream);
    dev_free(h->d_vel, h->last_stream);
    dev_free(h->d_status, h->last_stream);
    h->d_g.release();
    h->d_d.release();
    h->d_axes.release();
    h->d_partial.release();
    h->d_stat.release();
    h->d_best.release();
    h->d_cpart.release();
    h->d_clive.release();
    h->d_w.release();
    h->d_bank.release();
    h->d_selws.release();
    h->d_selzoom.release();
    dev_free(h->d_counter, h->last_stream);
    h->d_cw.release();
    progress_release(h->device, h->d_progress);
    h->d_sel.release();
    h->d_dts.release();
    h->d_dmm.release();
    h->d_slot.release();
    if (h->h_stage) cudaFreeHost(h->h_stage);
    if (h->ev_stage) cudaEventDestroy(h->ev_stage);
    for (auto &e : h->ev)
        if (e) cudaEventDestroy(e);
    delete h;
    return TCW_OK;
}

int tcw_set_option(tcw_handle *h, int key, long value)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    switch (key) {
    case TCW_OPT_KERNEL:
        if (value < 0 || value > 3) return fail(TCW_EINVAL, "TCW_OPT_KERNEL must be 0, 1, 2 or 3");
        h->opt_kernel = (int)value;
        return TCW_OK;
    case TCW_OPT_TIMING:
        if (value != 0 && value != 1) return fail(TCW_EINVAL, "TCW_OPT_TIMING must be 0 or 1");
        h->opt_timing = (int)value;
        h->timing_n = 0;
        return TCW_OK;
    case TCW_OPT_F0_PER_LANE:
        if (value != 0 && value != 4 && value != 8 && value != 16)
            return fail(TCW_EINVAL, "TCW_OPT_F0_PER_LANE must be 0, 4, 8 or 16");
        h->opt_r = (int)value;
        return TCW_OK;
    case TCW_OPT_STAGES:
        if (value != 0 && (value < 2 || value > 16)) return fail(TCW_EINVAL, "TCW_OPT_STAGES must be 0 or 2..16");
        h->opt_stages = (int)value;
        return TCW_OK;
    case TCW_OPT_SKY_BLOCK:
        if (value != 0 && value != 64 && value != 128 && value != 256)
            return fail(TCW_EINVAL, "TCW_OPT_SKY_BLOCK must be 0, 64, 128 or 256");
        h->opt_sky = (int)value;
        return TCW_OK;
    case TCW_OPT_EXACT_INDEX:
        if (value != 0 && value != 1) return fail(TCW_EINVAL, "TCW_OPT_EXACT_INDEX must be 0 or 1");
        h->opt_exact = (int)value;
        return TCW_OK;
    case TCW_OPT_GENERAL_F0:
        if (value != 0 && value != 1) return fail(TCW_EINVAL, "TCW_OPT_GENERAL_F0 must be 0 or 1");
        h->opt_nonuniform = (int)value;
        return TCW_OK;
    case TCW_OPT_ROW_COPIES:
        if (value != 0 && value != 1) return fail(TCW_EINVAL, "TCW_OPT_ROW_COPIES must be 0 or 1");
        h->opt_row_copies = (int)value;
        return TCW_OK;
    case TCW_OPT_DEBUG_SHRINK_SLOT:
        if (value < 0 || value > (1 << 20)) return fail(TCW_EINVAL, "TCW_OPT_DEBUG_SHRINK_SLOT must be 0..2^20");
        h->dbg_slot_shrink = (int)value;
        return TCW_OK;
    case TCW_OPT_DEBUG_CHUNK_SCRATCH:
        if (value < 0) return fail(TCW_EINVAL, "TCW_OPT_DEBUG_CHUNK_SCRATCH must be >= 0");
        h->chunk_scratch_max = value ? (double)value : CHUNK_SCRATCH_MAX;
        return TCW_OK;
    case TCW_OPT_DEBUG_FAIL_WAIT:
        if (value < 0 || value > 16) return fail(TCW_EINVAL, "TCW_OPT_DEBUG_FAIL_WAIT must be 0..16");
        h->dbg_fail_wait = (int)value;
        return TCW_OK;
    case TCW_OPT_CHUNK_ROWS:
        if (value < -1 || value > (1L << 30)) return fail(TCW_EINVAL, "TCW_OPT_CHUNK_ROWS must be -1, 0 or a row count");
        h->opt_chunk = value;
        return TCW_OK;
    default: return fail(TCW_EINVAL, "unknown option %d", key);
    }
}

// The search proper.  wt == NULL: the plain track sum (tcw_search).  Otherwise the weighted statistic,
// its critical ratio and the per-group maximum of the critical ratio (tcw_search_weighted).
static int search_impl(tcw_handle *h, const tcw_grid *grid, const tcw_weighting *wt, void *out_stat, float *out_psi,
                       void *out_best, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    int rc = validate_grid(h, grid);
    if (rc != TCW_OK) return rc;
    const bool wgt = wt != nullptr;
    if (!out_stat && !out_best && !out_psi) return fail(TCW_EINVAL, "every output pointer is NULL");
    if (wgt && (!std::isfinite(wt->mean1) || !(wt->var1 > 0) || !std::isfinite(wt->var1)))
        return fail(TCW_EINVAL, "weighting needs a finite mean1 and a finite var1 > 0");
    if (wgt && h->opt_kernel == 3)
        return fail(TCW_EUNSUPPORTED, "the sky-block kernel does not serve weighted searches (weights depend on the sky point)");
    cudaStream_t st = (cudaStream_t)stream;
    enter(h, st);
    const long n_groups = (long)grid->n_sky * grid->n_tau * grid->n_brk;
    if (!h->count_known) {
        // uint8 handle of tcw_create_async: the launch plan needs the largest count, so wait for the
        // upload and scan the rows now (tcw_create does this before returning)
        CUDA_TRY(cudaSetDevice(h->device));
        if (h->up_stream) CUDA_TRY(cudaStreamSynchronize(h->up_stream));
        int *d_max = nullptr;
        CUDA_TRY(dev_alloc((void **)&d_max, sizeof(int), st));
        CUDA_TRY(cudaMemsetAsync(d_max, 0, sizeof(int), st));
        tcw::max_u8_kernel<<<148 * 8, 256, 0, st>>>(h->d_spec + h->pad_bytes, h->pitch, h->n_sft, h->n_bins, d_max);
        CUDA_TRY(cudaGetLastError());
        CUDA_TRY(cudaMemcpyAsync(&h->count_max, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        dev_free(d_max, st);
        h->count_known = true;
    }

    tcw::SumParams p = base_params(h, grid);
    tcw::SkyParams q;
    std::memset(&q, 0, sizeof q);
    int kernel = 0, r = 0, stages = 0, slot = 0, sky_sc = 0, n_blocks = 0;
    size_t smem = 0;
    // ---- launch plan, count formats with many sky points: the sky-block kernel (tcw_skyblock.cuh)
    if (h->opt_kernel == 3 && h->fmt_dev != tcw::FMT_U8)
        return fail(TCW_EUNSUPPORTED, "the sky-block kernel serves the count formats only");
    if (!wgt && h->fmt_dev == tcw::FMT_U8 && (h->opt_kernel == 3 || (h->opt_kernel == 0 && grid->n_sky >= 16))) {
        // two sky points differ by |D_s - D_s'| <= 2 vmax / c whatever the block holds
        const double spread = grid->f0[grid->n_f0 - 1] * h->T * 2.0 * (h->vmax / C_LIGHT) * (1.0 + 1e-5);
        // two-level blocks of 256 sky points (tcw_skyblock2.cuh): the packed int16 corrections are exact while
        // n_sft * (largest count) < 2^15 (bit-packed input: counts are 0/1), and enough sky points to fill a block
        const bool can2 = (long)h->n_sft * std::max(h->count_max, 1) <= 32767;
        if (h->opt_sky == 256 && !can2)
            return fail(TCW_EUNSUPPORTED, "256-point sky blocks need n_sft * (largest count) <= 32767");
        if (can2 && (h->opt_sky == 256 || (h->opt_sky == 0 && grid->n_sky >= 128))) {
            const long w2 = max_window_bins(grid, tcw::F2, p.dmaxT) + (long)std::ceil(spread) + 2;
            const int sb2 = tcw::DTS2_BYTES + (int)((w2 + 32 + 15) & ~15L);
            if (w2 <= tcw::PAD_BINS && tcw::sky2_smem_bytes(sb2) <= SMEM_MAX) {
                kernel = 3; r = tcw::R2; sky_sc = 8; stages = tcw::D2; slot = sb2; smem = tcw::sky2_smem_bytes(sb2);
            }
        }
        const int sc = h->opt_sky == 128 ? 4 : 2, rr = sc == 2 ? 16 : 8, S = 32 * sc;
        const long w_bins = max_window_bins(grid, 32 * rr, p.dmaxT) + (long)std::ceil(spread) + 2;
        if (!kernel && w_bins <= tcw::PAD_BINS) {
            const int sb = 8 * S + (int)((w_bins + 32 + 15) & ~15L);
            for (int s = h->opt_stages ? std::min(h->opt_stages, 8) : 4; s >= 2; --s) {
                const size_t b = tcw::sky_smem_bytes(s, sb, 32 * rr, S);
                if (b <= SMEM_MAX) {
                    kernel = 3; r = rr; sky_sc = sc; stages = s; slot = sb; smem = b;
                    break;
                }
            }
        }
        if (!kernel && h->opt_kernel == 3)
            return fail(TCW_EUNSUPPORTED, "f0 spacing too wide for the sky-block kernel (window exceeds the row padding)");
    }
    // ---- otherwise: staged kernel with the largest tile whose window fits the row padding and
    // whose ring still lets 12 warps share an SM
    if (!kernel && h->opt_kernel != 1) {
        const int all[3] = {16, 8, 4};
        for (int c = 0; c < 3 && !kernel; ++c) {
            if (h->opt_r && all[c] != h->opt_r) continue;
            long w_bins = max_window_bins(grid, 32 * all[c], p.dmaxT);
            // equally spaced f0: the lanes past the end of a ragged last tile still form addresses (their sums
            // are discarded), so every slot holds the window of a whole tile
            if (p.d32 != 0.0)
                w_bins = std::max(w_bins, (long)std::floor((32 * all[c] - 1) * (p.d32 / 32.0) * p.dmaxT * (1.0 + 1e-9) + 1e-6) + 2);
            if (w_bins > tcw::PAD_BINS) continue;
            // one tensor-map copy per slot where the rows allow it
            const bool box = h->d_tmaps != nullptr && !h->opt_row_copies;
            if (!box) { p.tmaps = nullptr; p.max_seg = 0; }
            const int sb = slot_bytes_for(h->fmt_dev, w_bins, box);
            // rings holding at least six rows per warp (a slot is RB rows) hide the L2 latency; TCW_MINB CTAs of four warps per SM
            const int per_sm = TCW_MINB;
            for (int s = h->opt_stages ? std::min(h->opt_stages, 8) : (tcw::RB >= 4 ? 2 : 6 / tcw::RB); s >= 2; --s) {
                const size_t b = tcw::staged_smem_bytes(s, sb, 32 * all[c], wgt);
                if (b <= SMEM_MAX / per_sm - 1024 || (s == 2 && b <= SMEM_MAX)) {
                    kernel = 2; r = all[c]; stages = s; slot = sb; smem = b;
                    break;
                }
            }
        }
        if (!kernel && h->opt_kernel == 2)
            return fail(TCW_EUNSUPPORTED, "f0 spacing too wide for the staged kernel (window exceeds the row padding)");
    }
    if (!kernel) kernel = 1;
    p.tile = kernel >= 2 ? 32 * r : 128;
    p.n_tiles = (grid->n_f0 + p.tile - 1) / p.tile;
    p.stages = stages;
    p.slot_bytes = slot;
    p.slot_limit = slot - h->dbg_slot_shrink;   // = slot except under the test hook TCW_OPT_DEBUG_SHRINK_SLOT
    const long n_partial = n_groups * p.n_tiles;
    long n_ctas = n_partial;
    if (kernel == 2) {
        // SFT chunks (slowest block index): the CTAs in flight then share a set of rows small enough
        // to stay in L2 while every group reads it.  Only worth it when the rows do not fit anyway.
        const long rows = h->n_sft - p.j_begin;
        const double row_b = (double)(h->fmt_dev == tcw::FMT_F32 ? 4 : 1) * h->n_bins;
        long c_rows = 0;
        if (h->opt_chunk > 0) c_rows = h->opt_chunk;
        else if (h->opt_chunk == 0 && rows * row_b > CHUNK_MIN_BYTES) c_rows = std::min(CHUNK_MAX_ROWS, (long)(CHUNK_TARGET_BYTES / row_b));
        if (c_rows > 0) {
            c_rows = std::max<long>(64, (c_rows + 63) / 64 * 64);
            long nc = (rows + c_rows - 1) / c_rows;
            // The yes/no of chunking fixes the float32 summation order, so a group range (tcw_search_groups) must
            // decide it as the whole grid would: both size limits are tested on the whole grid's group count.  (A
            // range is never larger than its grid, so what the whole grid may chunk, the range may too.)
            const long plan_groups = std::max<long>(h->plan_groups, n_groups);
            const double scratch = (double)nc * (double)plan_groups * grid->n_f0 * (wgt ? 20.0 : 4.0);
            if (nc > 1 && nc <= 255 && scratch <= h->chunk_scratch_max && nc * (plan_groups * p.n_tiles) <= 2147483647L) {
                p.chunk_rows = (int)c_rows;
                p.n_chunks = (int)nc;
                n_ctas = nc * n_partial;
            }
        }
    }
    if (kernel == 3) {
        // sky points sorted by their Doppler shift at the middle SFT, cut into blocks of S
        const int S = 32 * sky_sc;
        n_blocks = (grid->n_sky + S - 1) / S;
        n_ctas = (long)n_blocks * p.n_ab * p.n_tiles;
        std::vector<std::pair<double, int>> key((size_t)grid->n_sky);
        for (int s = 0; s < grid->n_sky; ++s) {
            const double *n = grid->sky + 3 * (size_t)s;
            key[s] = {n[0] * h->vmid[0] + n[1] * h->vmid[1] + n[2] * h->vmid[2], s};
        }
        std::sort(key.begin(), key.end());
        h->slot_host.resize((size_t)n_blocks * S);
        for (size_t t = 0; t < h->slot_host.size(); ++t)
            h->slot_host[t] = key[std::min(t, (size_t)grid->n_sky - 1)].second;
    }
    if (n_ctas > 2147483647L) return fail(TCW_EUNSUPPORTED, "grid needs more than 2^31-1 CTAs; split the search");
    // progressive read-back (tcw_search_host): parts of the tau axis, CTAs issued part by part, one counter per part
    h->progress_active = false;
    if (h->want_parts > 1 && h->dl_ready && p.n_chunks == 1 && !wgt && !h->d_progress) h->d_progress = progress_acquire(h->device);
    if (h->want_parts > 1 && h->dl_ready && p.n_chunks == 1 && !wgt && h->d_progress) {
        const int np = std::min({h->want_parts, grid->n_tau, 16});
        const long units = kernel == 3 ? n_blocks : grid->n_sky;
        p.n_parts = np;
        h->progress_np = np;
        for (int r = 0; r <= np; ++r) {
            h->progress_a0[r] = (int)((long)grid->n_tau * r / np);
            p.part_ab0[r] = h->progress_a0[r] * grid->n_brk;
        }
        for (int r = 0; r < np; ++r)
            h->progress_target[r] = (unsigned int)(units * (p.part_ab0[r + 1] - p.part_ab0[r]) * p.n_tiles);
        CUDA_TRY(cudaSetDevice(h->device));
        CUDA_TRY(cudaMemsetAsync(h->d_progress, 0, 16 * sizeof(unsigned int), st));
        CUDA_TRY(cudaEventRecord(h->dl_ready, st));
        p.progress = h->d_progress;
        h->progress_active = true;
    }

    CUDA_TRY(cudaSetDevice(h->device));
    if ((rc = h->d_partial.reserve((size_t)n_partial * 8)) != TCW_OK) return rc;
    if (!out_best && (rc = h->d_best.reserve((size_t)n_groups * 8)) != TCW_OK) return rc;
    if (kernel == 3) {
        const size_t rows = (size_t)n_blocks * h->n_sft;
        if ((rc = h->d_dts.reserve(rows * (sky_sc == 8 ? (size_t)(tcw::DTS2_BYTES / 8) : (size_t)(32 * sky_sc)))) != TCW_OK) return rc;
        if ((rc = h->d_dmm.reserve(rows * 2)) != TCW_OK) return rc;
    }
    if (p.n_chunks > 1) {
        if ((rc = h->d_cpart.reserve((size_t)p.n_chunks * n_groups * grid->n_f0 * 4)) != TCW_OK) return rc;
        if ((rc = h->d_clive.reserve((size_t)p.n_chunks * n_partial)) != TCW_OK) return rc;
        p.cpart = h->d_cpart.p;
        p.clive = h->d_clive.p;
        if (wgt) {
            const size_t plane = (size_t)p.n_chunks * n_groups * grid->n_f0;
            if ((rc = h->d_cw.reserve(2 * plane)) != TCW_OK) return rc;
            p.cw1 = h->d_cw.p;
            p.cw2 = h->d_cw.p + plane;
        }
    }
    p.partial = h->d_partial.p;
    p.out_stat = out_stat;
    if (wgt) {
        p.mean1 = wt->mean1;
        p.var1 = wt->var1;
        p.out_psi = out_psi;
        if (wt->weights) {
            const size_t n_w = (size_t)grid->n_sky * h->n_sft;
            if ((rc = h->d_w.reserve(n_w)) != TCW_OK) return rc;
            CUDA_TRY(cudaMemcpyAsync(h->d_w.p, wt->weights, n_w * sizeof(float), cudaMemcpyDefault, st));
            p.wtab = h->d_w.p;
        }
    }

    const bool tm = h->opt_timing != 0 && h->timing_n < TIMING_MAX;
    cudaEvent_t *ev = nullptr;
    if (tm) {
        while (h->ev.size() < 4 * (h->timing_n + 1)) {
            cudaEvent_t e;
            CUDA_TRY(cudaEventCreate(&e));
            h->ev.push_back(e);
        }
        ev = h->ev.data() + 4 * h->timing_n;
        CUDA_TRY(cudaEventRecord(ev[0], st));
    }
    if (!h->keep_status) CUDA_TRY(cudaMemsetAsync(h->d_status, 0, sizeof(int), st));
    if ((rc = prepare(h, grid, 0, nullptr, st, kernel == 3 ? &h->slot_host : nullptr)) != TCW_OK) return rc;
    p.f0 = h->a_f0;
    p.gtab = h->d_g.p;
    p.dtab = h->d_d.p;
    if (kernel == 3) {
        if (sky_sc == 8) {
            const long warps = (long)n_blocks * h->n_sft;
            const unsigned blocks = (unsigned)((warps * 32 + 255) / 256);
            if (h->t_pow2)
                tcw::skyblock2_table_kernel<true><<<blocks, 256, 0, st>>>(h->d_vel, h->n_sft, h->a_sky, h->d_slot.p, n_blocks, h->T,
                                                                         h->d_dts.p, h->d_dmm.p);
            else
                tcw::skyblock2_table_kernel<false><<<blocks, 256, 0, st>>>(h->d_vel, h->n_sft, h->a_sky, h->d_slot.p, n_blocks, h->T,
                                                                          h->d_dts.p, h->d_dmm.p);
            CUDA_TRY(cudaGetLastError());
        } else if ((rc = launch_sky_table(sky_sc, h->t_pow2, h, h->a_sky, n_blocks, st)) != TCW_OK) return rc;
        q.dts = h->d_dts.p;
        q.dmm = h->d_dmm.p;
        q.slot_sky = h->d_slot.p;
        q.n_sky = grid->n_sky;
        q.n_blocks = n_blocks;
    }
    if (tm) CUDA_TRY(cudaEventRecord(ev[1], st));
    int extra_launches = 0;
    if (h->up_pending && kernel == 2 && p.n_chunks > 1) {
        // the spectrogram is still arriving (tcw_create_async): one launch per SFT chunk, each behind
        // the upload event of the chunk's last row, so the search overlaps the rest of the transfer
        for (int c = 0; c < p.n_chunks && rc == TCW_OK; ++c) {
            upload_wait_rows(h, std::min<long>(h->n_sft, (long)p.j_begin + (long)(c + 1) * p.chunk_rows), st);
            tcw::SumParams pc = p;
            pc.chunk0 = c;
            rc = launch_staged(h->fmt_dev, r, h->t_pow2, wgt, pc, n_partial, smem, st);
        }
        extra_launches = p.n_chunks - 1;
    } else {
        upload_wait_rows(h, h->n_sft, st);
        if (kernel == 3 && sky_sc == 8) {
            if (h->t_pow2) {
                CUDA_TRY(cudaFuncSetAttribute(tcw::sum_skyblock2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                tcw::sum_skyblock2_kernel<true><<<(unsigned)n_ctas, tcw::SKY2_THREADS, smem, st>>>(p, q);
            } else {
                CUDA_TRY(cudaFuncSetAttribute(tcw::sum_skyblock2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                tcw::sum_skyblock2_kernel<false><<<(unsigned)n_ctas, tcw::SKY2_THREADS, smem, st>>>(p, q);
            }
            CUDA_TRY(cudaGetLastError());
        } else if (kernel == 3) rc = launch_sky(sky_sc, h->t_pow2, p, q, n_ctas, smem, st);
        else if (kernel == 2) rc = launch_staged(h->fmt_dev, r, h->t_pow2, wgt, p, n_ctas, smem, st);
        else rc = launch_gather(h->fmt_dev, h->t_pow2, wgt, p, n_ctas, st);
    }
    if (rc != TCW_OK) return rc;
    upload_done(h, st);
    if (p.n_chunks > 1) {
        if (wgt) tcw::chunk_reduce_kernel<float, true><<<(unsigned)n_partial, 256, 0, st>>>(p);
        else if (h->format == TCW_F32_POWER) tcw::chunk_reduce_kernel<float, false><<<(unsigned)n_partial, 256, 0, st>>>(p);
        else tcw::chunk_reduce_kernel<int, false><<<(unsigned)n_partial, 256, 0, st>>>(p);
        CUDA_TRY(cudaGetLastError());
    }
    if (tm) CUDA_TRY(cudaEventRecord(ev[2], st));
    void *best_dst = out_best ? out_best : (void *)h->d_best.p;
    if (wgt || h->format == TCW_F32_POWER)
        tcw::best_kernel<float><<<(unsigned)((n_groups + 127) / 128), 128, 0, st>>>(
            (const tcw::Best<float> *)h->d_partial.p, n_groups, p.n_tiles, (tcw::Best<float> *)best_dst);
    else
        tcw::best_kernel<int><<<(unsigned)((n_groups + 127) / 128), 128, 0, st>>>(
            (const tcw::Best<int> *)h->d_partial.p, n_groups, p.n_tiles, (tcw::Best<int> *)best_dst);
    CUDA_TRY(cudaGetLastError());
    if (tm) {
        CUDA_TRY(cudaEventRecord(ev[3], st));
        h->timing_n++;
    }
    h->info[0] = kernel;
    h->info[1] = p.tile;
    h->info[2] = n_ctas;
    h->info[3] = (long)smem;
    h->info[6] = stages;
    h->info[7] = 32 * sky_sc;
    h->info[5] = (kernel == 3 ? 5 : 4) + (p.n_chunks > 1 ? 1 : 0) + extra_launches;  // doppler table, spin-down table, (sky-block table,) sum, (chunk reduce,) best
    h->info[8] = p.n_chunks;
    h->info[9] = p.chunk_rows;
    h->info[10] = h->progress_active ? h->progress_np : 0;
    h->info[11] = kernel == 2 && p.tmaps ? 1 : 0;     // the staged kernel may stage slots by tensor-map copies
    return TCW_OK;
}

int tcw_search(tcw_handle *h, const tcw_grid *grid, void *out_stat, void *out_best, void *stream)
{
    if (h && grid && !out_stat && !out_best) return fail(TCW_EINVAL, "out_stat and out_best are both NULL");
    return search_impl(h, grid, nullptr, out_stat, nullptr, out_best, stream);
}

int tcw_search_weighted(tcw_handle *h, const tcw_grid *grid, const tcw_weighting *weighting, float *out_psi,
                        float *out_stat, tcw_best_f32 *out_best, void *stream)
{
    if (h && !weighting) return fail(TCW_EINVAL, "weighting is NULL");
    return search_impl(h, grid, weighting, out_stat, out_psi, out_best, stream);
}

int tcw_search_bank(tcw_handle *h, const tcw_bank *bank, void *out_stat, int *out_inband, int *out_k, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    if (!bank) return fail(TCW_EINVAL, "bank is NULL");
    if (bank->n <= 0) return fail(TCW_EINVAL, "bank size must be positive");
    if (!bank->f0 || !bank->tau || !bank->brk || !bank->sky) return fail(TCW_EINVAL, "bank array pointer is NULL");
    if (!std::isfinite(bank->T0)) return fail(TCW_EINVAL, "T0 is not finite");
    if (!out_stat) return fail(TCW_EINVAL, "out_stat is NULL");
    const long n = bank->n;
    const double f_cap = (2147483648.0 - 1048576.0) / h->T;
    for (long q = 0; q < n; ++q) {
        if (!(bank->f0[q] > 0) || !(bank->f0[q] < f_cap)) return fail(TCW_EINVAL, "f0[%ld] must be > 0 and f0*T_sft < 2^31 - 2^20", q);
        if (!(bank->tau[q] > 0) || !std::isfinite(bank->tau[q])) return fail(TCW_EINVAL, "tau[%ld] must be > 0", q);
        if (!(bank->brk[q] > 1) || !std::isfinite(bank->brk[q])) return fail(TCW_EINVAL, "braking index brk[%ld] must be > 1", q);
    }
    const long n_vec = bank->sky_shared ? 1 : n;
    for (long q = 0; q < n_vec; ++q) {
        const double *v = bank->sky + 3 * q;
        const double nrm = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        if (!(std::fabs(nrm - 1.0) <= 1e-6)) return fail(TCW_EINVAL, "sky[%ld] is not a unit vector", q);
    }
    cudaStream_t st = (cudaStream_t)stream;
    enter(h, st);
    CUDA_TRY(cudaSetDevice(h->device));
    int rc;
    if ((rc = h->d_bank.reserve((size_t)(3 * n + 3 * n_vec))) != TCW_OK) return rc;
    if (bank->sky_shared && (rc = h->d_d.reserve((size_t)h->n_sft)) != TCW_OK) return rc;
    double *d_f0 = h->d_bank.p, *d_tau = d_f0 + n, *d_brk = d_tau + n, *d_sky = d_brk + n;
    CUDA_TRY(cudaMemcpyAsync(d_f0, bank->f0, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_tau, bank->tau, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_brk, bank->brk, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_sky, bank->sky, sizeof(double) * 3 * n_vec, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemsetAsync(h->d_counter, 0, sizeof(unsigned long long), st));
    // every search starts with a clear status word (tcw.h: tcw_check reports on the LAST search, bank searches included)
    if (!h->keep_status) CUDA_TRY(cudaMemsetAsync(h->d_status, 0, sizeof(int), st));

    const bool tm = h->opt_timing != 0 && h->timing_n < TIMING_MAX;
    cudaEvent_t *ev = nullptr;
    if (tm) {
        while (h->ev.size() < 4 * (h->timing_n + 1)) {
            cudaEvent_t e;
            CUDA_TRY(cudaEventCreate(&e));
            h->ev.push_back(e);
        }
        ev = h->ev.data() + 4 * h->timing_n;
        CUDA_TRY(cudaEventRecord(ev[0], st));
    }
    if (bank->sky_shared) {
        // the exact Doppler factor of the shared sky point, one entry per SFT (eq. (2))
        tcw::doppler_table_kernel<<<(unsigned)((h->n_sft + 255) / 256), 256, 0, st>>>(h->d_vel, h->n_sft, d_sky, 1, h->d_d.p);
        CUDA_TRY(cudaGetLastError());
    }
    if (tm) CUDA_TRY(cudaEventRecord(ev[1], st));
    tcw::BankParams p;
    std::memset(&p, 0, sizeof p);
    p.spec = h->d_spec + h->pad_bytes;
    p.pitch = h->pitch;
    p.n_sft = h->n_sft;
    p.n_bins = h->n_bins;
    p.k_min = h->k_min;
    p.j_begin = (int)(std::lower_bound(h->ts.begin(), h->ts.end(), bank->T0) - h->ts.begin());
    p.T = h->T;
    p.T0 = bank->T0;
    p.ts = h->d_ts;
    p.vel = h->d_vel;
    p.dshared = bank->sky_shared ? h->d_d.p : nullptr;
    p.n_tpl = n;
    p.f0 = d_f0;
    p.tau = d_tau;
    p.brk = d_brk;
    p.sky = d_sky;
    p.dmax = (1.0 + (h->vmax / C_LIGHT) * (1.0 + 1e-5) + 1e-15) * (1.0 + 1e-9);
    p.out_stat = out_stat;
    p.out_inband = out_inband;
    p.out_k = out_k;
    p.n_exact = h->d_counter;
    const long n_ctas = (n + tcw::BANK_THREADS - 1) / tcw::BANK_THREADS;
    if (n_ctas > 2147483647L) return fail(TCW_EUNSUPPORTED, "bank needs more than 2^31-1 CTAs; split the search");
    upload_wait_rows(h, h->n_sft, st);
    upload_done(h, st);
    if (h->fmt_dev == tcw::FMT_F32) {
        if (h->t_pow2) tcw::sum_bank_kernel<tcw::FMT_F32, true><<<(unsigned)n_ctas, tcw::BANK_THREADS, 0, st>>>(p);
        else tcw::sum_bank_kernel<tcw::FMT_F32, false><<<(unsigned)n_ctas, tcw::BANK_THREADS, 0, st>>>(p);
    } else {
        if (h->t_pow2) tcw::sum_bank_kernel<tcw::FMT_U8, true><<<(unsigned)n_ctas, tcw::BANK_THREADS, 0, st>>>(p);
        else tcw::sum_bank_kernel<tcw::FMT_U8, false><<<(unsigned)n_ctas, tcw::BANK_THREADS, 0, st>>>(p);
    }
    CUDA_TRY(cudaGetLastError());
    if (tm) {
        CUDA_TRY(cudaEventRecord(ev[2], st));
        CUDA_TRY(cudaEventRecord(ev[3], st));
        h->timing_n++;
    }
    h->last_stream = st;
    h->tab_tau = 0;   // the grid tables of an earlier search are gone (d_d is reused)
    h->info[0] = 4;
    h->info[1] = tcw::BANK_THREADS;
    h->info[2] = n_ctas;
    h->info[3] = 0;
    h->info[5] = bank->sky_shared ? 2 : 1;
    h->info[6] = 0;
    h->info[7] = 0;
    h->info[8] = 1;
    h->info[9] = h->n_sft;
    return TCW_OK;
}

int tcw_get_counter(tcw_handle *h, int which, long long *value)
{
    if (!h || !value) return fail(TCW_EINVAL, "NULL argument");
    if (which != 0) return fail(TCW_EINVAL, "unknown counter %d", which);
    CUDA_TRY(cudaSetDevice(h->device));
    if (h->last_stream || h->info[0]) CUDA_TRY(cudaStreamSynchronize(h->last_stream));
    unsigned long long v = 0;
    CUDA_TRY(cudaMemcpy(&v, h->d_counter, sizeof v, cudaMemcpyDeviceToHost));
    *value = (long long)v;
    return TCW_OK;
}

namespace {
struct SelScratch {
    unsigned int *hist, *blk_gt, *blk_eq, *cand_bits;
    unsigned long long *off_gt, *off_eq;
    long long *cand_idx;
    tcw::SelState *state;
};

int sel_scratch(tcw_handle *h, SelScratch *sc)
{
    const size_t B = tcw::SEL_MAX_BLOCKS, K = tcw::SEL_MAX_K;
    const size_t bytes = 2048 * 4 + 256 + 2 * B * 4 + 2 * B * 8 + K * 4 + K * 8;
    int rc = h->d_selws.reserve(bytes);
    if (rc != TCW_OK) return rc;
    unsigned char *q = h->d_selws.p;
    sc->off_gt = (unsigned long long *)q; q += B * 8;
    sc->off_eq = (unsigned long long *)q; q += B * 8;
    sc->cand_idx = (long long *)q; q += K * 8;
    sc->state = (tcw::SelState *)q; q += 256;
    sc->hist = (unsigned int *)q; q += 2048 * 4;
    sc->blk_gt = (unsigned int *)q; q += B * 4;
    sc->blk_eq = (unsigned int *)q; q += B * 4;
    sc->cand_bits = (unsigned int *)q;
    return TCW_OK;
}

// contiguous segment per CTA (a multiple of the CTA size), at most SEL_MAX_BLOCKS CTAs
void sel_grid(long n, long *seg, int *n_blocks)
{
    long want = std::min<long>(tcw::SEL_MAX_BLOCKS, std::max<long>(1, (n + 8191) / 8192));
    long s = (n + want - 1) / want;
    s = (s + 2 * tcw::SEL_TILE - 1) / (2 * tcw::SEL_TILE) * (2 * tcw::SEL_TILE);   // whole tile pairs: 16-byte aligned starts
    *seg = s;
    *n_blocks = (int)((n + s - 1) / s);
}
}  // namespace

int tcw_topk(tcw_handle *h, const void *values, int dtype, long n, int K, void *out_val, long long *out_idx,
             int *out_count, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    if (!values || !out_val || !out_idx) return fail(TCW_EINVAL, "NULL array pointer");
    if (dtype != 0 && dtype != 1) return fail(TCW_EINVAL, "dtype must be 0 (float32) or 1 (int32)");
    if (n <= 0) return fail(TCW_EINVAL, "n must be positive");
    if (K <= 0 || K > tcw::SEL_MAX_K) return fail(TCW_EINVAL, "K must be in 1..%d", tcw::SEL_MAX_K);
    if (n >= (1L << 32)) return fail(TCW_EUNSUPPORTED, "n must be below 2^32 (the selection counters are 32-bit)");
    cudaStream_t st = (cudaStream_t)stream;
    enter(h, st);
    CUDA_TRY(cudaSetDevice(h->device));
    SelScratch sc;
    int rc = sel_scratch(h, &sc);
    if (rc != TCW_OK) return rc;
    const unsigned int *v = (const unsigned int *)values;
    CUDA_TRY(cudaMemsetAsync(sc.hist, 0, 2048 * 4, st));
    CUDA_TRY(cudaMemsetAsync(sc.state, 0, sizeof(tcw::SelState), st));
    // the exact selection over `vals` (radix select of the K-th key, ordered compaction, sort); see sel_gate for `gate`
    auto run_select = [&](const unsigned int *vals, long nn, int gate, const long long *idx_map) {
        long seg;
        int nb;
        sel_grid(nn, &seg, &nb);
        const int vec = ((uintptr_t)vals & 15) == 0;
        tcw::sel_hist_kernel<0><<<nb, tcw::SEL_THREADS, 0, st>>>(vals, nn, seg, dtype, vec, sc.state, sc.hist, gate);
        tcw::sel_pick_kernel<0><<<1, 256, 0, st>>>(sc.hist, sc.state, (unsigned int)K, gate);
        tcw::sel_hist_kernel<1><<<nb, tcw::SEL_THREADS, 0, st>>>(vals, nn, seg, dtype, vec, sc.state, sc.hist, gate);
        tcw::sel_pick_kernel<1><<<1, 256, 0, st>>>(sc.hist, sc.state, (unsigned int)K, gate);
        tcw::sel_hist_kernel<2><<<nb, tcw::SEL_THREADS, 0, st>>>(vals, nn, seg, dtype, vec, sc.state, sc.hist, gate);
        tcw::sel_pick_kernel<2><<<1, 256, 0, st>>>(sc.hist, sc.state, (unsigned int)K, gate);
        tcw::sel_count_kernel<false><<<nb, tcw::SEL_THREADS, 0, st>>>(vals, nn, seg, dtype, vec, sc.state, 0.0, sc.blk_gt, sc.blk_eq, gate);
        tcw::sel_scan_kernel<<<1, 256, 0, st>>>(sc.blk_gt, sc.blk_eq, nb, sc.off_gt, sc.off_eq, sc.state, gate);
        tcw::sel_scatter_kernel<false><<<nb, tcw::SEL_THREADS, 0, st>>>(vals, nn, seg, dtype, vec, sc.state, 0.0, sc.blk_gt, sc.blk_eq,
                                                                        sc.off_gt, sc.off_eq, 0, sc.cand_bits, sc.cand_idx, idx_map, gate);
        tcw::sel_sort_kernel<<<1, 1024, 0, st>>>(sc.cand_bits, sc.cand_idx, dtype, sc.state, (unsigned int *)out_val, out_idx,
                                                 out_count, gate);
    };
    if (n >= TOPK_TWO_READ_MIN) {
        // two reads of the array: zoomed histogram (+ per-CTA histograms), then ordered compaction of the keys at or
        // above the bin of the K-th largest into a candidate buffer; the exact selection then runs on the candidates
        // (gate 2), or, if they did not fit (heavily tied data), on the full array (gate 1).  No host synchronisation.
        long seg;
        int nb;
        sel_grid(n, &seg, &nb);
        const int vec = ((uintptr_t)values & 15) == 0;
        const size_t n_rows = (size_t)((n + tcw::SEL_ROW - 1) / tcw::SEL_ROW);
        const size_t zbytes = (size_t)nb * 2048 * 4 + 2 * (size_t)tcw::SEL_MAX_BLOCKS * 4 + (size_t)tcw::SEL_MAX_CAND * 12 + 64 + n_rows * 2;
        if ((rc = h->d_selzoom.reserve(zbytes)) != TCW_OK) return rc;
        long long *z_idx = (long long *)h->d_selzoom.p;
        unsigned int *z_bits = (unsigned int *)(z_idx + tcw::SEL_MAX_CAND);
        unsigned int *z_off = z_bits + tcw::SEL_MAX_CAND;
        unsigned int *z_cnt = z_off + tcw::SEL_MAX_BLOCKS;
        unsigned int *z_hist = z_cnt + tcw::SEL_MAX_BLOCKS;
        unsigned short *z_rows = (unsigned short *)(z_hist + (size_t)nb * 2048);      // largest zoom bin of every row of 128 values
        CUDA_TRY(cudaMemsetAsync(z_rows, 0, n_rows * 2, st));
        tcw::sel_sample_kernel<<<1, 1024, 0, st>>>(v, n, dtype, (unsigned int)K, sc.state);
        if (dtype) tcw::sel_zoom_hist_kernel<1><<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, vec, sc.state, sc.hist, z_hist, z_rows);
        else tcw::sel_zoom_hist_kernel<0><<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, vec, sc.state, sc.hist, z_hist, z_rows);
        tcw::sel_zoom_pick_kernel<<<1, 256, 0, st>>>(sc.hist, sc.state, (unsigned int)K, dtype);
        tcw::sel_zoom_count_kernel<<<(nb + 7) / 8, 256, 0, st>>>(z_hist, nb, sc.state, z_cnt);
        tcw::sel_zoom_scan_kernel<<<1, 256, 0, st>>>(z_cnt, nb, z_off);
        if (dtype) tcw::sel_zoom_compact_kernel<1><<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, vec, sc.state, z_off, z_rows, z_bits, z_idx);
        else tcw::sel_zoom_compact_kernel<0><<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, vec, sc.state, z_off, z_rows, z_bits, z_idx);
        run_select(z_bits, tcw::SEL_MAX_CAND, 2, z_idx);
        run_select(v, n, 1, nullptr);
    } else {
        run_select(v, n, 0, nullptr);
    }
    CUDA_TRY(cudaGetLastError());
    h->last_stream = st;
    return TCW_OK;
}

int tcw_select_above(tcw_handle *h, const void *values, int dtype, long n, double threshold, long capacity,
                     long long *out_idx, long long *out_count, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    if (!values || !out_count || (capacity > 0 && !out_idx)) return fail(TCW_EINVAL, "NULL array pointer");
    if (dtype != 0 && dtype != 1) return fail(TCW_EINVAL, "dtype must be 0 (float32) or 1 (int32)");
    if (n <= 0 || capacity < 0) return fail(TCW_EINVAL, "n must be positive and capacity >= 0");
    if (std::isnan(threshold)) return fail(TCW_EINVAL, "threshold is NaN");
    if (n >= (1L << 32)) return fail(TCW_EUNSUPPORTED, "n must be below 2^32 (the per-block counters are 32-bit)");
    cudaStream_t st = (cudaStream_t)stream;
    enter(h, st);
    CUDA_TRY(cudaSetDevice(h->device));
    SelScratch sc;
    int rc = sel_scratch(h, &sc);
    if (rc != TCW_OK) return rc;
    long seg;
    int nb;
    sel_grid(n, &seg, &nb);
    const unsigned int *v = (const unsigned int *)values;
    const int vec = ((uintptr_t)values & 15) == 0;
    // the count pass leaves, per row of 128 values, how many are selected (n/128 bytes); the scatter pass opens only those rows
    const size_t n_rows = (size_t)((n + tcw::SEL_ROW - 1) / tcw::SEL_ROW);
    if ((rc = h->d_selzoom.reserve(n_rows)) != TCW_OK) return rc;
    unsigned char *row_cnt = (unsigned char *)h->d_selzoom.p;
    CUDA_TRY(cudaMemsetAsync(row_cnt, 0, n_rows, st));
    tcw::sel_count_kernel<true><<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, dtype, vec, sc.state, threshold, sc.blk_gt, sc.blk_eq, 0, row_cnt);
    tcw::sel_scan_kernel<<<1, 256, 0, st>>>(sc.blk_gt, sc.blk_eq, nb, sc.off_gt, sc.off_eq, sc.state);
    if (capacity > 0)
        tcw::sel_scatter_rows_kernel<<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, dtype, vec, threshold, row_cnt, sc.off_gt, capacity, out_idx);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(out_count, &sc.state->count, sizeof(long long), cudaMemcpyDeviceToDevice, st));
    h->last_stream = st;
    return TCW_OK;
}

// ---- tcw_select_above_static: the threshold selection with its scratch inside the library image ---------
// For callers that cannot let a library allocate (a job that filled the GPU with its own arrays, a host
// program whose allocator owns the device memory, a loop that must not take the device-wide synchronisation of
// cudaMalloc / cudaFree while searches run on other streams): include/tcw.h has the contract.  The scratch that
// tcw_select_above takes from the handle is here one file-scope device array, laid out as
//   [SSEL_OFF_GT]  off_gt   SEL_MAX_BLOCKS x u64    exclusive scan of the per-CTA hit counts
//   [SSEL_OFF_EQ]  off_eq   SEL_MAX_BLOCKS x u64    (written by the shared scan kernel, unused by this selection)
//   [SSEL_STATE]   SelState 256 bytes               .count = total hits
//   [SSEL_BLK_GT]  blk_gt   SEL_MAX_BLOCKS x u32    hits per CTA, every launched CTA writes its entry
//   [SSEL_BLK_EQ]  blk_eq   SEL_MAX_BLOCKS x u32
//   [SSEL_ROWS]    row_cnt  one byte per row of SEL_ROW values: must be ZERO where no value is selected, and
//                           the count kernel writes only rows that hold a hit -> cleared on every call
// Every GPU that loads the library carries the array (SSEL_BYTES, about 2.1 MB) until the process exits.
namespace {
constexpr size_t SSEL_OFF_GT = 0;
constexpr size_t SSEL_OFF_EQ = SSEL_OFF_GT + (size_t)tcw::SEL_MAX_BLOCKS * 8;
constexpr size_t SSEL_STATE = SSEL_OFF_EQ + (size_t)tcw::SEL_MAX_BLOCKS * 8;
constexpr size_t SSEL_BLK_GT = SSEL_STATE + 256;
constexpr size_t SSEL_BLK_EQ = SSEL_BLK_GT + (size_t)tcw::SEL_MAX_BLOCKS * 4;
constexpr size_t SSEL_ROWS = SSEL_BLK_EQ + (size_t)tcw::SEL_MAX_BLOCKS * 4;
constexpr size_t SSEL_MAX_ROWS = (size_t)(TCW_SELECT_STATIC_MAX_N / tcw::SEL_ROW);
constexpr size_t SSEL_BYTES = SSEL_ROWS + SSEL_MAX_ROWS;
static_assert(sizeof(tcw::SelState) <= 256 && SSEL_ROWS % 256 == 0 && TCW_SELECT_STATIC_MAX_N % tcw::SEL_ROW == 0,
              "static selection scratch layout");
}  // namespace

static __device__ __align__(256) unsigned char g_static_select_scratch[SSEL_BYTES];

namespace {
// In host code `g_static_select_scratch` is only the host-side handle of the symbol, not an address a kernel can
// use: the device address differs per GPU and comes from cudaGetSymbolAddress with that GPU current.  Looked up
// once per device and kept (the lookup allocates nothing; it may load the module, hence "before stream capture").
int static_select_scratch(unsigned char **out)
{
    static std::mutex mu;
    static unsigned char *ptr[64];
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(TCW_EUNSUPPORTED, "device ordinal %d is outside 0..63", dev);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void *p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, g_static_select_scratch));
        if (!p) return fail(TCW_ECUDA, "cudaGetSymbolAddress gave a NULL address for the static selection scratch");
        ptr[dev] = (unsigned char *)p;
    }
    *out = ptr[dev];
    return TCW_OK;
}
}  // namespace

int tcw_select_above_static(const void *values, int dtype, long n, double threshold, long capacity, long long *out_idx,
                            long long *out_count, void *stream)
{
    if (!values || !out_count || (capacity > 0 && !out_idx)) return fail(TCW_EINVAL, "NULL array pointer");
    if (dtype != 0 && dtype != 1) return fail(TCW_EINVAL, "dtype must be 0 (float32) or 1 (int32)");
    if (n <= 0 || capacity < 0) return fail(TCW_EINVAL, "n must be positive and capacity >= 0");
    if (std::isnan(threshold)) return fail(TCW_EINVAL, "threshold is NaN");
    if (n > TCW_SELECT_STATIC_MAX_N)
        return fail(TCW_EUNSUPPORTED, "n = %ld exceeds TCW_SELECT_STATIC_MAX_N = %ld, the size the library's built-in scratch "
                    "covers; use tcw_select_above (scratch from a handle) for larger arrays", n, (long)TCW_SELECT_STATIC_MAX_N);
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *base = nullptr;
    int rc = static_select_scratch(&base);
    if (rc != TCW_OK) return rc;
    unsigned long long *off_gt = (unsigned long long *)(base + SSEL_OFF_GT), *off_eq = (unsigned long long *)(base + SSEL_OFF_EQ);
    tcw::SelState *state = (tcw::SelState *)(base + SSEL_STATE);
    unsigned int *blk_gt = (unsigned int *)(base + SSEL_BLK_GT), *blk_eq = (unsigned int *)(base + SSEL_BLK_EQ);
    unsigned char *row_cnt = base + SSEL_ROWS;
    long seg;
    int nb;
    sel_grid(n, &seg, &nb);
    const unsigned int *v = (const unsigned int *)values;
    const int vec = ((uintptr_t)values & 15) == 0;
    const size_t n_rows = (size_t)((n + tcw::SEL_ROW - 1) / tcw::SEL_ROW);
    // the previous call's row counts are still there: clear the rows this call covers (everything else in the
    // array is written before it is read: blk_* by every CTA of the count pass, off_* and state->count by the scan)
    CUDA_TRY(cudaMemsetAsync(row_cnt, 0, n_rows, st));
    tcw::sel_count_kernel<true><<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, dtype, vec, state, threshold, blk_gt, blk_eq, 0, row_cnt);
    tcw::sel_scan_kernel<<<1, 256, 0, st>>>(blk_gt, blk_eq, nb, off_gt, off_eq, state);
    if (capacity > 0)
        tcw::sel_scatter_rows_kernel<<<nb, tcw::SEL_THREADS, 0, st>>>(v, n, seg, dtype, vec, threshold, row_cnt, off_gt, capacity, out_idx);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(out_count, &state->count, sizeof(long long), cudaMemcpyDeviceToDevice, st));
    return TCW_OK;
}

int tcw_prepare(const float *strain, long n_samples, const tcw_prep *prep, int format, void *out_spectrogram,
                long out_pitch_bytes, int *n_sft, void *stream)
{
    if (!strain || !prep || !out_spectrogram || !n_sft) return fail(TCW_EINVAL, "NULL argument");
    if (format != TCW_F32_POWER && format != TCW_U8_COUNT && format != TCW_BIT_COUNT)
        return fail(TCW_EINVAL, "unknown spectrogram format %d", format);
    if (!(prep->fs > 0) || !(prep->T_sft > 0) || !std::isfinite(prep->fs) || !std::isfinite(prep->T_sft))
        return fail(TCW_EINVAL, "fs and T_sft must be positive");
    const double Nd = std::rint(prep->fs * prep->T_sft);
    if (std::fabs(prep->fs * prep->T_sft - Nd) > 1e-9 || Nd < 2 || Nd > (double)(1 << 27) || ((long)Nd & 1))
        return fail(TCW_EINVAL, "fs*T_sft must be an even integer number of samples (2..2^27)");
    const int N = (int)Nd, n_half = N / 2 + 1;
    const long n_seg = n_samples / N;
    if (n_seg <= 0 || n_seg > 2147483647L) return fail(TCW_EINVAL, "n_samples holds no whole segment (or too many)");
    const int W = prep->median_bins, h = (W - 1) / 2;
    if (W < 1 || W > tcw::PREP_MAX_W || !(W & 1)) return fail(TCW_EINVAL, "median_bins must be odd, 1..%d", tcw::PREP_MAX_W);
    const double km = std::rint(prep->f_min * prep->T_sft);
    if (!(prep->f_min >= 0) || std::fabs(prep->f_min * prep->T_sft - km) > 1e-9)
        return fail(TCW_EINVAL, "f_min*T_sft must be a non-negative integer (bin-aligned band start)");
    if (prep->n_bins <= 0 || km - h < 0 || km + prep->n_bins + h > n_half)
        return fail(TCW_EINVAL, "band plus median half-window does not fit the bins 0..N/2");
    if (format != TCW_F32_POWER && std::isnan(prep->threshold)) return fail(TCW_EINVAL, "threshold is NaN");
    if (out_pitch_bytes < (long)row_bytes(format, prep->n_bins) || (format != TCW_U8_COUNT && (out_pitch_bytes & 3)))
        return fail(TCW_EINVAL, "out_pitch_bytes is smaller than one row or not a multiple of 4");
    int spc = tcw::PREP_SPC;                        // SFTs per CTA: as many as leave room for two CTAs per SM
    while (spc > 1 && spc * tcw::prep_sft_smem(prep->n_bins, h) > SMEM_MAX / 2 - 1024) spc /= 2;
    const size_t smem = spc * tcw::prep_sft_smem(prep->n_bins, h);
    if (smem > SMEM_MAX) return fail(TCW_EUNSUPPORTED, "band too wide for one CTA's shared memory (%zu bytes)", smem);

    cudaStream_t st = (cudaStream_t)stream;
    // Transforms run in batches whose samples (64 MB) stay in L2 between the window kernel and cuFFT; their spectra
    // are kept for a SUPER-batch of up to 2 GiB (16 384 eight-second SFTs at 4096 Hz) and normalised by ONE launch:
    // a batch of 512 SFTs is only 128 CTAs (fewer than the 148 SMs, eight warps each), and a kernel whose threads
    // each walk a long dependent loop needs the whole machine full of warps.
    const int batch = (int)std::min<long>(n_seg, std::max<long>(1, (64L << 20) / ((long)N * 4)));
    const long super = std::min<long>(n_seg, std::max<long>(batch, ((2L << 30) / ((long)n_half * 8)) / batch * batch));
    float *d_x = nullptr, *d_win = nullptr;
    float2 *d_spec = nullptr;
    cufftHandle plan = 0;
    // a device-resident strain is windowed straight out of the caller's buffer; a host one is staged
    cudaPointerAttributes attr;
    const bool on_device = cudaPointerGetAttributes(&attr, strain) == cudaSuccess &&
                           (attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged);
    cudaGetLastError();   // a plain host pointer may leave an error state on older runtimes
    int rc = TCW_OK;
#define PREP_TRY(call)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            rc = fail(e_ == cudaErrorMemoryAllocation ? TCW_ENOMEM : TCW_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
            goto done;                                                                              \
        }                                                                                           \
    } while (0)
    PREP_TRY(dev_alloc((void **)&d_x, (size_t)batch * N * sizeof(float), st));
    PREP_TRY(dev_alloc((void **)&d_spec, (size_t)(super + batch) * n_half * sizeof(float2), st));   // + batch: cuFFT always writes whole batches
    PREP_TRY(dev_alloc((void **)&d_win, (size_t)N * sizeof(float), st));
    tcw::prep_window_table_kernel<<<(N + 255) / 256, 256, 0, st>>>(N, d_win);
    PREP_TRY(cudaGetLastError());
    {
        // one cached plan per thread (device, N, batch): creating a plan costs more than transforming a day of data
        struct PlanCache { cufftHandle plan; int dev, N, batch; bool ok; };
        static thread_local PlanCache pc = {0, -1, 0, 0, false};
        int dev = 0;
        cudaGetDevice(&dev);
        if (!pc.ok || pc.dev != dev || pc.N != N || pc.batch != batch) {
            if (pc.ok) cufftDestroy(pc.plan);
            pc.ok = false;
            int dims[1] = {N};
            if (cufftPlanMany(&pc.plan, 1, dims, nullptr, 1, N, nullptr, 1, n_half, CUFFT_R2C, batch) != CUFFT_SUCCESS) {
                rc = fail(TCW_ECUDA, "cufftPlanMany failed");
                goto done;
            }
            pc.dev = dev; pc.N = N; pc.batch = batch; pc.ok = true;
        }
        plan = pc.plan;
        if (cufftSetStream(plan, st) != CUFFT_SUCCESS) { rc = fail(TCW_ECUDA, "cufftSetStream failed"); goto done; }
    }
    PREP_TRY(cudaFuncSetAttribute(tcw::prep_normalise_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    for (long s0 = 0; s0 < n_seg; s0 += super) {
        const long ns = std::min<long>(super, n_seg - s0);
        for (long j0 = s0; j0 < s0 + ns; j0 += batch) {
            const int nb = (int)std::min<long>(batch, s0 + ns - j0);
            if (nb < batch)   // zero the tail of the batch buffer: cuFFT always transforms `batch` segments
                PREP_TRY(cudaMemsetAsync(d_x + (size_t)nb * N, 0, (size_t)(batch - nb) * N * sizeof(float), st));
            if (!on_device)
                PREP_TRY(cudaMemcpyAsync(d_x, strain + j0 * N, (size_t)nb * N * sizeof(float), cudaMemcpyHostToDevice, st));
            {
                const float *src = on_device ? strain + j0 * N : d_x;
                if ((N & 3) == 0 && ((uintptr_t)src & 15) == 0)
                    tcw::prep_window4_kernel<<<dim3((unsigned)((N / 4 + 255) / 256), (unsigned)std::min(nb, 64)), 256, 0, st>>>(src, d_win, nb, N, d_x);
                else
                    tcw::prep_window_kernel<<<148 * 8, 256, 0, st>>>(src, d_win, nb, N, d_x);
            }
            PREP_TRY(cudaGetLastError());
            if (cufftExecR2C(plan, d_x, (cufftComplex *)(d_spec + (size_t)(j0 - s0) * n_half)) != CUFFT_SUCCESS) { rc = fail(TCW_ECUDA, "cufftExecR2C failed"); goto done; }
        }
        tcw::PrepParams p;
        p.spec = d_spec;
        p.n_half = n_half;
        p.k_min = (int)km;
        p.n_bins = prep->n_bins;
        p.h = h;
        p.threshold = (float)prep->threshold;
        p.out_format = format;
        p.out = (unsigned char *)out_spectrogram + s0 * out_pitch_bytes;
        p.out_pitch = out_pitch_bytes;
        tcw::prep_normalise_kernel<<<(unsigned)((ns + spc - 1) / spc), tcw::PREP_THREADS, smem, st>>>(p, (int)ns, spc);
        PREP_TRY(cudaGetLastError());
    }
    PREP_TRY(cudaStreamSynchronize(st));
    *n_sft = (int)n_seg;
done:
#undef PREP_TRY
    dev_free(d_x, st);
    dev_free(d_win, st);
    dev_free(d_spec, st);
    return rc;
}

// A contiguous range [g0, g1) of the flattened group index (s*n_tau + a)*n_brk + b as at most seven
// sub-grids, in ascending group order; the output of each (its own [s][a][b][f0] layout) is then a
// contiguous slice of the full output: whole sky points, whole tau rows of one sky point, or part
// of one tau row.
struct GroupRect { int s0, s1, a0, a1, b0, b1; };
static std::vector<GroupRect> split_groups(int n_tau, int n_brk, long g0, long g1)
{
    std::vector<GroupRect> out;
    const long per_sky = (long)n_tau * n_brk;
    long cur = g0;
    while (cur < g1) {
        const long s = cur / per_sky, rem = cur % per_sky;
        if (rem == 0 && g1 - cur >= per_sky) {
            const long ns = (g1 - cur) / per_sky;
            out.push_back({(int)s, (int)(s + ns), 0, n_tau, 0, n_brk});
            cur += ns * per_sky;
            continue;
        }
        const long e = std::min(g1, (s + 1) * per_sky) - s * per_sky;   // end of the range inside sky point s
        const int a = (int)(rem / n_brk), b = (int)(rem % n_brk);
        if (b != 0 || e - rem < n_brk) {
            const int b1 = (int)std::min<long>(n_brk, b + (e - rem));
            out.push_back({(int)s, (int)s + 1, a, a + 1, b, b1});
            cur += b1 - b;
        } else {
            const int na = (int)((e - rem) / n_brk);
            out.push_back({(int)s, (int)s + 1, a, a + na, 0, n_brk});
            cur += (long)na * n_brk;
        }
    }
    return out;
}

static tcw_grid sub_grid(const tcw_grid *g, const GroupRect &r)
{
    tcw_grid s = *g;
    s.n_sky = r.s1 - r.s0; s.sky = g->sky + 3 * (size_t)r.s0;
    s.n_tau = r.a1 - r.a0; s.tau = g->tau + r.a0;
    s.n_brk = r.b1 - r.b0; s.brk = g->brk + r.b0;
    return s;
}

int tcw_split_groups(int n_tau, int n_brk, long group_begin, long group_end, int rects[7][6], int *n_rects)
{
    if (!rects || !n_rects) return fail(TCW_EINVAL, "NULL argument");
    if (n_tau <= 0 || n_brk <= 0 || group_begin < 0 || group_begin > group_end)
        return fail(TCW_EINVAL, "sizes must be positive and the range ordered");
    const std::vector<GroupRect> v = split_groups(n_tau, n_brk, group_begin, group_end);
    if (v.size() > 7) return fail(TCW_EINTERNAL, "group range split into %zu rectangles", v.size());
    for (size_t i = 0; i < v.size(); ++i) {
        const int r[6] = {v[i].s0, v[i].s1, v[i].a0, v[i].a1, v[i].b0, v[i].b1};
        std::memcpy(rects[i], r, sizeof r);
    }
    *n_rects = (int)v.size();
    return TCW_OK;
}

int tcw_search_groups(tcw_handle *h, const tcw_grid *grid, long group_begin, long group_end, void *out_stat,
                      void *out_best, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    int rc = validate_grid(h, grid);
    if (rc != TCW_OK) return rc;
    if (!out_stat && !out_best) return fail(TCW_EINVAL, "out_stat and out_best are both NULL");
    const long n_groups = (long)grid->n_sky * grid->n_tau * grid->n_brk;
    if (group_begin < 0 || group_end > n_groups || group_begin >= group_end)
        return fail(TCW_EINVAL, "group range [%ld, %ld) is empty or outside 0..%ld", group_begin, group_end, n_groups);
    cudaStream_t st = (cudaStream_t)stream;
    enter(h, st);
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaMemsetAsync(h->d_status, 0, sizeof(int), st));
    h->keep_status = true;
    h->plan_groups = n_groups;
    long info_sum[3] = {0, 0, 0};   // CTAs, kernels launched, parts
    for (const GroupRect &r : split_groups(grid->n_tau, grid->n_brk, group_begin, group_end)) {
        const tcw_grid sub = sub_grid(grid, r);
        const long first = ((long)r.s0 * grid->n_tau + r.a0) * grid->n_brk + r.b0 - group_begin;
        rc = search_impl(h, &sub, nullptr, out_stat ? (char *)out_stat + (size_t)first * grid->n_f0 * 4 : nullptr, nullptr,
                         out_best ? (char *)out_best + (size_t)first * 8 : nullptr, stream);
        if (rc != TCW_OK) break;
        info_sum[0] += h->info[2]; info_sum[1] += h->info[5]; info_sum[2]++;
    }
    h->keep_status = false;
    h->plan_groups = 0;
    if (rc == TCW_OK) { h->info[2] = info_sum[0]; h->info[5] = info_sum[1]; }
    return rc;
}

// Outputs of at least this many bytes are read back part by part (tau sub-ranges) while the next part is searched.
constexpr size_t HOST_OVERLAP_MIN_BYTES = 64u << 20, HOST_PART_BYTES = 40u << 20;

int tcw_search_host(tcw_handle *h, const tcw_grid *grid, void *out_stat_host, void *out_best_host, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    int rc = validate_grid(h, grid);
    if (rc != TCW_OK) return rc;
    if (!out_stat_host && !out_best_host) return fail(TCW_EINVAL, "out_stat and out_best are both NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n_groups = (size_t)grid->n_sky * grid->n_tau * grid->n_brk;
    const size_t n_templates = n_groups * grid->n_f0;
    enter(h, st);
    CUDA_TRY(cudaSetDevice(h->device));
    if (out_stat_host && (rc = h->d_stat.reserve(n_templates * 4)) != TCW_OK) return rc;
    if ((rc = h->d_best.reserve(n_groups * 8)) != TCW_OK) return rc;
    int n_parts = 1;
    if (out_stat_host && n_templates * 4 >= HOST_OVERLAP_MIN_BYTES)
        n_parts = (int)std::min<size_t>({(size_t)grid->n_tau, (n_templates * 4 + HOST_PART_BYTES / 2) / HOST_PART_BYTES, (size_t)16});
    if (n_parts <= 1) {
        rc = tcw_search(h, grid, out_stat_host ? (void *)h->d_stat.p : nullptr, h->d_best.p, stream);
        if (rc != TCW_OK) return rc;
        if (out_stat_host)
            CUDA_TRY(cudaMemcpyAsync(out_stat_host, h->d_stat.p, n_templates * 4, cudaMemcpyDeviceToHost, st));
        if (out_best_host)
            CUDA_TRY(cudaMemcpyAsync(out_best_host, h->d_best.p, n_groups * 8, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        return check_status(h);
    }
    // Large outputs: ONE search whose CTAs are issued tau range by tau range and count themselves done per
    // range (SumParams::progress); the read-back stream waits for each counter (cuStreamWaitValue32) and
    // copies that range -- n_sky rows of the [sky][tau][brk][f0] layout, one strided copy -- while the later
    // ranges are still being searched.  No launch is split, so no wave is left half empty.
    typedef CUresult (*wait_value_fn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
    static wait_value_fn wait_value = [] {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            fn = nullptr;
        cudaGetLastError();
        return (wait_value_fn)fn;
    }();
    if (!h->dl_stream) CUDA_TRY(cudaStreamCreateWithFlags(&h->dl_stream, cudaStreamNonBlocking));
    if (!h->dl_ready) CUDA_TRY(cudaEventCreateWithFlags(&h->dl_ready, cudaEventDisableTiming));
    h->want_parts = wait_value ? n_parts : 0;
    rc = tcw_search(h, grid, h->d_stat.p, h->d_best.p, stream);
    h->want_parts = 0;
    if (rc != TCW_OK) return rc;
    const size_t row_t = (size_t)grid->n_brk * grid->n_f0 * 4;   // bytes per (sky, tau)
    const size_t pitch_t = (size_t)grid->n_tau * row_t;
    if (h->progress_active) {
        cudaError_t e = cudaStreamWaitEvent(h->dl_stream, h->dl_ready, 0);     // the counters have been cleared
        int p_plain = h->progress_np;      // parts from here on go back by plain copies on the search stream
        for (int p = 0; p < h->progress_np && e == cudaSuccess; ++p) {
            const int a0 = h->progress_a0[p], a1 = h->progress_a0[p + 1];     // np <= n_tau: never empty
            const CUresult wr = h->dbg_fail_wait == p + 1 ? CUDA_ERROR_NOT_SUPPORTED :
                wait_value((CUstream)h->dl_stream, (CUdeviceptr)(h->d_progress + p), h->progress_target[p], CU_STREAM_WAIT_VALUE_GEQ);
            if (wr != CUDA_SUCCESS) {
                // the driver refuses the stream wait (e.g. CUDA_ERROR_NOT_SUPPORTED): the search itself is fine, so the
                // remaining ranges are copied after it, in stream order; the waits already queued are satisfied by the
                // running search as usual
                p_plain = p;
                break;
            }
            e = cudaMemcpy2DAsync((char *)out_stat_host + (size_t)a0 * row_t, pitch_t, h->d_stat.p + (size_t)a0 * row_t, pitch_t,
                                  (size_t)(a1 - a0) * row_t, (size_t)grid->n_sky, cudaMemcpyDeviceToHost, h->dl_stream);
        }
        if (e == cudaSuccess && p_plain < h->progress_np) {
            const int a0 = h->progress_a0[p_plain], a1 = h->progress_a0[h->progress_np];
            e = cudaMemcpy2DAsync((char *)out_stat_host + (size_t)a0 * row_t, pitch_t, h->d_stat.p + (size_t)a0 * row_t, pitch_t,
                                  (size_t)(a1 - a0) * row_t, (size_t)grid->n_sky, cudaMemcpyDeviceToHost, st);
        }
        h->info[10] = p_plain;             // parts that really went back under the search
        if (e != cudaSuccess) {
            rc = fail(TCW_ECUDA, "progressive read-back: %s", cudaGetErrorString(e));
            // Waits already queued on dl_stream must not be left hanging.  CU_STREAM_WAIT_VALUE_GEQ is the cyclic
            // compare (int32)(*addr - value) >= 0, so the value that releases a wait is its own target (0xffffffff
            // would not: target - 1 steps "behind").  Let the search finish, then write every target.
            cudaStreamSynchronize(st);
            cudaMemcpyAsync(h->d_progress, h->progress_target, (size_t)h->progress_np * sizeof(unsigned int), cudaMemcpyHostToDevice, st);
            cudaStreamSynchronize(st);
            cudaStreamSynchronize(h->dl_stream);
            return rc;
        }
    } else {
        CUDA_TRY(cudaMemcpyAsync(out_stat_host, h->d_stat.p, n_templates * 4, cudaMemcpyDeviceToHost, st));
    }
    if (out_best_host)
        CUDA_TRY(cudaMemcpyAsync(out_best_host, h->d_best.p, n_groups * 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaStreamSynchronize(h->dl_stream));
    return check_status(h);
}

int tcw_measure_peaks(double *out, int n_out, void *stream)
{
    if (!out || n_out < 10) return fail(TCW_EINVAL, "out must hold 10 doubles");
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, n_sm = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    float *d_out = nullptr;
    CUDA_TRY(cudaMalloc((void **)&d_out, 64));
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    const int ctas = n_sm * 8, iters = 4096;
    const double warps = (double)ctas * (tcw::PEAK_THREADS / 32);
    int rc = TCW_OK;
    // each measurement: one warm-up launch, then the best of three timed launches
    auto timed = [&](auto launch, double work, double *rate) {
        launch();
        float best = 1e30f;
        for (int rep = 0; rep < 3; ++rep) {
            cudaEventRecord(e0, st);
            launch();
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = fail(TCW_ECUDA, "peak kernel: %s", cudaGetErrorString(cudaGetLastError())); return; }
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            best = std::min(best, ms);
        }
        *rate = work / (best * 1e-3);
    };
    const double fp64_inst = warps * iters * 4.0 * tcw::PEAK_ILP;
    timed([&] { tcw::peak_fp64_kernel<0><<<ctas, tcw::PEAK_THREADS, 0, st>>>(iters, 1.0, (double *)d_out); }, fp64_inst, &out[0]);
    timed([&] { tcw::peak_fp64_kernel<1><<<ctas, tcw::PEAK_THREADS, 0, st>>>(iters, 1.0, (double *)d_out); }, fp64_inst, &out[1]);
    timed([&] { tcw::peak_fp64_kernel<2><<<ctas, tcw::PEAK_THREADS, 0, st>>>(iters, 1.0, (double *)d_out); }, fp64_inst, &out[2]);
    timed([&] { tcw::peak_issue_kernel<<<ctas, tcw::PEAK_THREADS, 0, st>>>(4 * iters, 1.0f, d_out); }, 4.0 * fp64_inst, &out[3]);
    timed([&] { tcw::peak_lds_kernel<<<ctas, tcw::PEAK_THREADS, 0, st>>>(iters, d_out); }, warps * iters * 16.0, &out[4]);
    {
        const int rows = 8192, c_ctas = n_sm * 3 * 4;
        // y = dlane*c + r*4c + q stays inside [1.5*2^20 + 8, 1.5*2^20 + 640)
        timed([&] { tcw::peak_chain_kernel<<<c_ctas, 128, 0, st>>>(rows, 0.93, 1572864.0 + 8.5, d_out); },
              (double)c_ctas * 128.0 * rows * 16.0, &out[5]);
    }
    {
        const int rows = 8192, c_ctas = n_sm * 3 * 4;
        const double work = (double)c_ctas * 128.0 * rows * 16.0;
        timed([&] { tcw::peak_count_chain_kernel<false><<<c_ctas, 128, 0, st>>>(rows, 0.93, 1572864.0 + 8.5, (int *)d_out); }, work, &out[8]);
        timed([&] { tcw::peak_count_chain_kernel<true><<<c_ctas, 128, 0, st>>>(rows, 0.93, 1572864.0 + 8.5, (int *)d_out); }, work, &out[9]);
    }
    if (n_out >= 12) {
        // staging alone (peak_stage_kernel): 2048 rows of a 20 000-bin float32 band, 2080-byte windows
        out[10] = out[11] = 0.0;
        const long pitch = 81920 + 8448;
        const int n_rows = 2048, slots = 128, c_ctas = n_sm * 3 * 8;
        unsigned char *d_arr = nullptr, *d_maps = nullptr;
        const size_t smem = 128 + (size_t)4 * 2 * tcw::RB * tcw::PEAK_STAGE_ROW;
        if (cudaMalloc((void **)&d_arr, (size_t)pitch * n_rows) == cudaSuccess) {
            cudaMemsetAsync(d_arr, 1, (size_t)pitch * n_rows, st);
            cudaFuncSetAttribute(tcw::peak_stage_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaFuncSetAttribute(tcw::peak_stage_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            const double n_slots = (double)c_ctas * 4 * slots;
            timed([&] { tcw::peak_stage_kernel<false><<<c_ctas, 128, smem, st>>>(d_arr, pitch, n_rows, slots, 2080, nullptr, 0, (unsigned *)d_out); },
                  n_slots * tcw::RB * 2080.0, &out[10]);
            std::vector<CUtensorMap> maps;
            if (encode_box_maps(d_arr, pitch, n_rows, maps) && cudaMalloc((void **)&d_maps, maps.size() * sizeof(CUtensorMap)) == cudaSuccess) {
                cudaMemcpy(d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice);
                timed([&] { tcw::peak_stage_kernel<true><<<c_ctas, 128, smem, st>>>(d_arr, pitch, n_rows, slots, 0, d_maps, 17, (unsigned *)d_out); },
                      n_slots * tcw::RB * 17.0 * 128.0, &out[11]);
            }
            cudaStreamSynchronize(st);
            cudaFree(d_maps);
            cudaFree(d_arr);
        }
        cudaGetLastError();
    }
    out[6] = (double)n_sm;
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    out[7] = (double)khz * 1e3;     // the device's nominal maximum SM clock (Hz)
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    if (rc == TCW_OK) CUDA_TRY(cudaGetLastError());
    return rc;
}

int tcw_check(tcw_handle *h)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaStreamSynchronize(h->last_stream));
    return check_status(h);
}

int tcw_track_indices(tcw_handle *h, const tcw_grid *grid, long n_sel, const long *sel, int *out_k, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    int rc = validate_grid(h, grid);
    if (rc != TCW_OK) return rc;
    if (n_sel <= 0 || !sel || !out_k) return fail(TCW_EINVAL, "selection is empty or NULL");
    const long n_templates = (long)grid->n_sky * grid->n_tau * grid->n_brk * grid->n_f0;
    for (long q = 0; q < n_sel; ++q)
        if (sel[q] < 0 || sel[q] >= n_templates) return fail(TCW_EINVAL, "sel[%ld] is not a template index", q);
    cudaStream_t st = (cudaStream_t)stream;
    enter(h, st);
    if ((rc = prepare(h, grid, n_sel, sel, st)) != TCW_OK) return rc;
    tcw::SumParams p = base_params(h, grid);
    const long total = n_sel * h->n_sft;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (h->t_pow2) tcw::track_index_kernel<true><<<blocks, 256, 0, st>>>(p, h->d_sel.p, n_sel, p.n_ab, out_k);
    else tcw::track_index_kernel<false><<<blocks, 256, 0, st>>>(p, h->d_sel.p, n_sel, p.n_ab, out_k);
    CUDA_TRY(cudaGetLastError());
    return TCW_OK;
}

int tcw_tables(tcw_handle *h, double *out_g, double *out_d, void *stream)
{
    if (!h) return fail(TCW_EINVAL, "handle is NULL");
    if (!h->tab_tau) return fail(TCW_EINVAL, "no search has been run on this handle");
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(cudaSetDevice(h->device));
    if (out_g)
        CUDA_TRY(cudaMemcpyAsync(out_g, h->d_g.p, sizeof(double) * (size_t)h->tab_tau * h->tab_brk * h->n_sft,
                                 cudaMemcpyDeviceToHost, st));
    if (out_d)
        CUDA_TRY(cudaMemcpyAsync(out_d, h->d_d.p, sizeof(double) * (size_t)h->tab_sky * h->n_sft,
                                 cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return TCW_OK;
}

int tcw_get_timing(tcw_handle *h, float ms[4], int *n_searches)
{
    if (!h || !ms) return fail(TCW_EINVAL, "NULL argument");
    if (!h->timing_n) return fail(TCW_EINVAL, "no timed search: set TCW_OPT_TIMING = 1 before tcw_search");
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaEventSynchronize(h->ev[4 * h->timing_n - 1]));
    double acc[4] = {0, 0, 0, 0};
    for (size_t q = 0; q < h->timing_n; ++q) {
        const cudaEvent_t *e = h->ev.data() + 4 * q;
        float t[4];
        CUDA_TRY(cudaEventElapsedTime(&t[0], e[0], e[1]));
        CUDA_TRY(cudaEventElapsedTime(&t[1], e[1], e[2]));
        CUDA_TRY(cudaEventElapsedTime(&t[2], e[2], e[3]));
        CUDA_TRY(cudaEventElapsedTime(&t[3], e[0], e[3]));
        for (int c = 0; c < 4; ++c) acc[c] += t[c];
    }
    for (int c = 0; c < 4; ++c) ms[c] = (float)(acc[c] / (double)h->timing_n);
    if (n_searches) *n_searches = (int)h->timing_n;
    h->timing_n = 0;
    return check_status(h);   // the last timed search has completed: times of an invalid search are an error
}

int tcw_get_info(tcw_handle *h, long info[12])
{
    if (!h || !info) return fail(TCW_EINVAL, "NULL argument");
    if (!h->info[0]) return fail(TCW_EINVAL, "no search has been run on this handle");
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaStreamSynchronize(h->last_stream));
    const int rc = check_status(h);
    std::memcpy(info, h->info, sizeof h->info);   // filled either way: info[4] holds the status word
    return rc;
}

}  // extern "C"
