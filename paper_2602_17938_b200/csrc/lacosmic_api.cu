// C-ABI boundary of liblacosmic_b200.so: argument checks, workspace carve-up, kernel sequence.
// See include/lacosmic.h for the contract of every entry point.
#include "../../include/lacosmic.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "kernels.cuh"
#include "lazy.cuh"
#include "grow.cuh"
#include "select.cuh"
#include "selectz.cuh"
#include "compact.cuh"
#include "probe.cuh"
#include "sepmed.cuh"

namespace {

thread_local int g_last_cuda_error = 0;
thread_local int g_launches = 0;
thread_local bool g_stats = false;   // lacosmic_stats_enable: per-iteration work counters for bench.py's roofline terms

inline bool cuda_ok(cudaError_t e) {
    if (e != cudaSuccess) {
        g_last_cuda_error = (int)e;
        return false;
    }
    return true;
}
#define CK(expr) do { if (!cuda_ok(expr)) return LACOSMIC_ERR_CUDA; } while (0)
#define LAUNCHED() do { ++g_launches; if (!cuda_ok(cudaGetLastError())) return LACOSMIC_ERR_CUDA; } while (0)

// Launch of a kernel of the lazy frame with programmatic dependent launch (common.cuh, pdl_entry): the grid may be
// scheduled while its predecessor in the stream drains; the kernel itself waits for the predecessor before it reads
// anything.  LACOSMIC_PDL=0 in the environment launches plainly.
std::atomic<int> g_pdl{-1};   // -1: not decided yet; two threads deciding at once store the same value
bool pdl_enabled() {
    int v = g_pdl.load(std::memory_order_relaxed);
    if (v < 0) {
        const char* e = std::getenv("LACOSMIC_PDL");
        v = (e && e[0] == '0') ? 0 : 1;
        g_pdl.store(v, std::memory_order_relaxed);
    }
    return v == 1;
}
template <class... KArgs, class... Args>
void launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    // not inside a stream capture: the replayed graph is faster with plain kernel-to-kernel edges (measured on B200:
    // 0.589 ms per frame replayed without the attribute, 0.603 with it; launched directly 0.616 without, 0.604 with)
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    const bool capturing = cudaStreamIsCapturing(st, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone;
    cfg.numAttrs = (pdl_enabled() && !capturing) ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// Optional per-kernel-class CUDA-event timing (lacosmic_kernel_timing_*): bench.py switches it on to
// measure the dominant kernel's average launch duration on the launching stream.
enum KClass { KC_NOISE_S = 0, KC_FINE_GATES, KC_GROW, KC_LISTS, KC_BITS, KC_EVAL, KC_NOISE_S_QUADS, KC_SELECT, KC_STEP, KC_COUNT };
static_assert(KC_COUNT == LACOSMIC_NUM_KERNEL_CLASSES, "header and library disagree");
struct KTiming {
    static constexpr int MAXSPANS = 8192;
    bool enabled = false;
    int n = 0;
    cudaEvent_t* ev = nullptr;   // 2 * MAXSPANS events, created on first enable
    int cls[MAXSPANS];
};
thread_local KTiming g_kt;

struct Span {   // records an event pair around one launch when timing is enabled
    int i = -1;
    cudaStream_t st;
    Span(int cls, cudaStream_t s) : st(s) {
        if (g_kt.enabled && g_kt.n < KTiming::MAXSPANS) {
            i = g_kt.n++;
            g_kt.cls[i] = cls;
            cudaEventRecord(g_kt.ev[2 * i], st);
        }
    }
    ~Span() {
        if (i >= 0) cudaEventRecord(g_kt.ev[2 * i + 1], st);
    }
};

// ---- TMA descriptors and persistent-grid sizing -------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            return nullptr;
        return (EncodeTiledFn)p;
    }();
    return fn;
}

// 2-D map over a row-major fp32 [h][w] plane (w % 4 == 0), box = boxW x boxH elements, zero fill
// outside; elements are moved as raw 32-bit words.
bool make_map(CUtensorMap* m, const float* base, int h, int w, int boxW, int boxH) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {(cuuint64_t)w, (cuuint64_t)h};
    cuuint64_t strides[1] = {(cuuint64_t)w * 4};
    cuuint32_t box[2] = {(cuuint32_t)boxW, (cuuint32_t)boxH};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, (void*)base, dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

#ifndef LAC_NS_WAVES
#define LAC_NS_WAVES 8
#endif
#ifndef LAC_FG_WAVES
#define LAC_FG_WAVES 6
#endif
struct DeviceInfo {
    int sms = 0, occ_noise = 0, occ_fine = 0, occ_quads = 0, occ_eval = 0, occ_rounds = 0;
    bool ok = false;
};

// Per-device: the SM count, the occupancy of the persistent kernels and the opt-in to > 48 KB of dynamic shared
// memory (a per-device function attribute) belong to the CURRENT device, which may differ from call to call.
constexpr int MAX_DEVICES = 64;
DeviceInfo device_info() {
    static DeviceInfo infos[MAX_DEVICES];
    static std::mutex mu;
    const DeviceInfo bad;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return bad;
    std::lock_guard<std::mutex> lock(mu);
    DeviceInfo& d = infos[dev];
    if (d.ok) return d;
    d = DeviceInfo();
    if (cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return d;
    if (cudaFuncSetAttribute(lac::k_fine_gates_tma, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             lac::FG_SMEM_BYTES) != cudaSuccess) return d;
    if (cudaFuncSetAttribute(lac::k_noise_S_tma<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, lac::NS_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(lac::k_noise_S_tma<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, lac::NS_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(lac::k_noise_S_tma<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, lac::NS_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(lac::k_noise_S_tma<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, lac::NS_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(lac::k_noise_S_tma<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, lac::NS_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(lac::k_noise_S_tma<9>, cudaFuncAttributeMaxDynamicSharedMemorySize, lac::NS_SMEM_BYTES) != cudaSuccess)
        return d;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&d.occ_fine, lac::k_fine_gates_tma, lac::NT,
                                                      lac::FG_SMEM_BYTES) != cudaSuccess) return d;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&d.occ_noise, lac::k_noise_S_tma<3>, lac::NT,
                                                      lac::NS_SMEM_BYTES) != cudaSuccess) return d;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&d.occ_quads, lac::k_noise_S_quads, 256, 0) != cudaSuccess) return d;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&d.occ_eval, lac::k_eval_candidates<0>, 128, 0) != cudaSuccess) return d;
    // gain estimate: the grid of the cooperative k_sel_rounds must be resident as a whole; clusters of 16 CTAs
    // (k_selz_resolve) are a non-portable size
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&d.occ_rounds, lac::k_sel_rounds, 256, 0) != cudaSuccess) return d;
    if (lac::SELZ_CLUSTER > 8 &&
        cudaFuncSetAttribute(lac::k_selz_resolve, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) return d;
    d.ok = d.sms > 0 && d.occ_fine > 0 && d.occ_noise > 0 && d.occ_quads > 0 && d.occ_eval > 0 && d.occ_rounds > 0;
    return d;
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline int words_per_row(int w) { return (w + 31) / 32; }

inline int check_shape(int h, int w) {
    if (h < 1 || w < 1) return LACOSMIC_ERR_SHAPE;
    if ((long long)h * (long long)w >= (1LL << 31)) return LACOSMIC_ERR_SHAPE;
    return LACOSMIC_OK;
}

inline int check_params(const lacosmic_params& p) {
    if (!std::isfinite(p.gain) || !std::isfinite(p.readnoise) || !std::isfinite(p.sigclip) ||
        !std::isfinite(p.sigfrac) || !std::isfinite(p.objlim) || std::isnan(p.satlevel))
        return LACOSMIC_ERR_PARAM;
    if (!(p.gain >= 0.0f) || p.readnoise < 0.0f || !(p.sigclip > 0.0f) || !(p.sigfrac > 0.0f) ||
        p.sigfrac > 1.0f || p.objlim < 0.0f || p.niter < 0 || p.niter > LACOSMIC_MAX_NITER)
        return LACOSMIC_ERR_PARAM;
    if (p.mode != LACOSMIC_MODE_LAZY && p.mode != LACOSMIC_MODE_DENSE) return LACOSMIC_ERR_PARAM;
    return LACOSMIC_OK;
}

inline bool overlap(const void* a, size_t na, const void* b, size_t nb) {
    uintptr_t pa = (uintptr_t)a, pb = (uintptr_t)b;
    return pa < pb + nb && pb < pa + na;
}

// Workspace layout (all offsets 256-byte aligned)
struct Workspace {
    float* S;          // significance plane; persistent across the iterations of a frame
    int32_t* clist;    // compacted candidate pixel list (capacity h*w)
    int32_t* qlist;    // compacted quad list of the incremental noise/S pass (capacity h*ceil(w/4))
    uint32_t *G1, *G2, *G2F, *M1, *M2, *M3, *C[2], *A1, *A2, *NEED;
    uint32_t *NOK, *DONX;  // R23 / R25: pixels never flagged (bad pixels | extended saturated-star mask); bad pixels
    int32_t* counts;   // per iteration: newly flagged pixels
    int32_t* ncand;    // per iteration (lazy path): candidate pixels evaluated
    int32_t* nquad;    // per iteration (lazy path): quads the incremental noise/S pass recomputed
    int32_t *nneed, *nfine;   // per iteration, only with lacosmic_stats_enable: replacement values computed; fine tests
    float* gains;      // per iteration: the gain the noise model used (R21: estimated when p.gain == 0)
    lac::SelState* sel; // radix selection state and histogram of the gain estimation (select.cuh)
    uint32_t* hist;
    lac::SelZone* zone; // fast path of the gain estimation (selectz.cuh): plan, bucket counts, zone id of every bucket
    uint32_t *histz, *histm;
    size_t bytes;      // total
    size_t zero_off, zero_bytes;   // region cleared at the start of a frame: the counters
};
constexpr int NCOUNTERS = LACOSMIC_NUM_FRAME_STATS * LACOSMIC_MAX_NITER;

Workspace carve(void* base, int h, int w) {
    Workspace ws;
    size_t P = (size_t)h * w, plane = align_up(P * 4, 256);
    size_t bp = align_up((size_t)h * words_per_row(w) * 4, 256);
    char* p = (char*)base;
    size_t off = 0;
    ws.S = (float*)(p + off); off += plane;
    ws.clist = (int32_t*)(p + off); off += plane;
    ws.qlist = (int32_t*)(p + off); off += align_up((size_t)h * ((w + 3) / 4) * 4, 256);
    uint32_t** planes[] = {&ws.G1, &ws.G2, &ws.G2F, &ws.M1, &ws.M2, &ws.M3, &ws.C[0], &ws.C[1], &ws.A1, &ws.A2, &ws.NEED,
                           &ws.NOK, &ws.DONX};
    for (uint32_t** pl : planes) { *pl = (uint32_t*)(p + off); off += bp; }
    ws.zero_off = off;
    ws.counts = (int32_t*)(p + off); off += align_up(NCOUNTERS * 4, 256);
    ws.ncand = ws.counts + LACOSMIC_MAX_NITER;
    ws.nquad = ws.counts + 2 * LACOSMIC_MAX_NITER;
    ws.nneed = ws.counts + 3 * LACOSMIC_MAX_NITER;
    ws.nfine = ws.counts + 4 * LACOSMIC_MAX_NITER;
    ws.gains = (float*)(p + off); off += align_up(LACOSMIC_MAX_NITER * 4, 256);
    ws.sel = (lac::SelState*)(p + off); off += 256;
    ws.hist = (uint32_t*)(p + off); off += align_up(lac::SEL_BINS * 4, 256);
    ws.zone = (lac::SelZone*)(p + off); off += align_up(sizeof(lac::SelZone), 256);
    ws.histz = (uint32_t*)(p + off); off += align_up(lac::SELZ_NB * 4, 256);
    ws.histm = (uint32_t*)(p + off); off += align_up(lac::SELZ_NB * 4, 256);
    ws.zero_bytes = off - ws.zero_off;
    ws.bytes = off;
    return ws;
}

int unpack(const uint32_t* bits, uint8_t* u8, int h, int w, cudaStream_t st, const int* counts_src = nullptr,
           int* counts_dst = nullptr, int ncounts = 0) {
    const unsigned g = (unsigned)(((size_t)h * w / 16 + 1 + 255) / 256);   // one thread per aligned 16 bytes (+ head)
    Span sp(KC_BITS, st);
    lac::k_unpack_bits<<<g, 256, 0, st>>>(bits, u8, h, w, words_per_row(w), counts_src, counts_dst, ncounts);
    LAUNCHED();
    return LACOSMIC_OK;
}

// grid of the bit-plane list kernels: 32 words x 64 rows per CTA (common.cuh)
// (1-D grids of nbx * nby CTAs, block_xy in common.cuh: rows on gridDim.y would stop at 65535 rows of CTAs)
inline int bit_nbx(int w) { return (words_per_row(w) + 31) / 32; }
inline unsigned bit_grid(int h, int w) { return (unsigned)bit_nbx(w) * (unsigned)((h + lac::BW_CTA_ROWS - 1) / lac::BW_CTA_ROWS); }
// grid of k_grow_replace / k_dirty_lists: 30 words x WG_R * WG_WARPS = 32 rows per CTA, one 30-word x 4-row strip per warp (grow.cuh)
inline int grow_nbx(int w) { return (words_per_row(w) + lac::WG_OWN - 1) / lac::WG_OWN; }
inline unsigned grow_grid(int h, int w) {
    const int rows = lac::WG_R * lac::WG_WARPS;
    return (unsigned)grow_nbx(w) * (unsigned)((h + rows - 1) / rows);
}

// steps (6)-(7) of one iteration, fused (grow.cuh)
int grow_replace(const lac::GrowArgs& ga, const int* prev, cudaStream_t st) {
    Span sp(KC_GROW, st);
    launch_pdl(lac::k_grow_replace, dim3(grow_grid(ga.h, ga.w)), dim3(32 * lac::WG_WARPS), 0, st, ga, prev);
    LAUNCHED();
    return LACOSMIC_OK;
}

// R21: sigma clipping of the residual plane R, typical signal from the med5 plane M5 (select.cuh, selectz.cuh)
// -> *gain_out (device), stats (nullable, device, 7 floats).  `lists`: storage of the fast path's lists (list_words
// 32-bit words: the quad list and the planes G1, G2, G2F, M1, M2, M3 behind it, which hold nothing at this point of an
// iteration that estimates the gain -- such an iteration is never incremental and rewrites them all).
std::atomic<int> g_gain_fast{-1};   // -1: not decided yet (environment LACOSMIC_GAIN_FAST=0 switches the fast path off)
bool gain_fast_enabled() {
    int v = g_gain_fast.load(std::memory_order_relaxed);
    if (v < 0) {
        const char* e = std::getenv("LACOSMIC_GAIN_FAST");
        v = (e && e[0] == '0') ? 0 : 1;
        int expect = -1;
        if (!g_gain_fast.compare_exchange_strong(expect, v)) v = expect;   // lacosmic_gain_fast_path_enable got there first
    }
    return v == 1;
}
int sigma_clip_gain(const float* R, const float* M5, size_t npx, const Workspace& ws, void* lists, size_t list_words,
                    float rn2, float* gain_out, float* stats, const int* prev, cudaStream_t st) {
    const DeviceInfo di = device_info();
    if (!di.ok) { g_last_cuda_error = (int)cudaGetLastError(); return LACOSMIC_ERR_CUDA; }
    const int sms = di.sms;
#ifndef LAC_SEL_CTAS_PER_SM
#define LAC_SEL_CTAS_PER_SM 8
#endif
    // full occupancy measured best on B200 (8 > 4 > 2 > 1 CTAs per SM): the pass is a streaming read
    const int grid = (int)std::min<size_t>((size_t)sms * LAC_SEL_CTAS_PER_SM, (npx / 4 + 255) / 256 + 1);
    // the lists of the fast path (selectz.cuh) live in the quad list's storage
    const float2* olist = lac::selz_carve(lists, list_words).o;
    const int grid_h = (int)std::min<size_t>((size_t)sms, (npx / 4 + 4 * lac::SELZ_HT - 1) / (4 * lac::SELZ_HT) + 1);
    Span sp(KC_SELECT, st);
    lac::k_selz_init<<<1, lac::SELZ_IT, 0, st>>>(R, M5, npx, ws.sel, ws.zone, ws.hist, ws.histz, ws.histm,
                                                     gain_fast_enabled() ? 0 : 1, prev);
    LAUNCHED();
    lac::k_selz_hist<<<grid_h, lac::SELZ_HT, 0, st>>>(R, M5, npx, ws.sel, ws.zone, ws.histz, ws.histm, lists, list_words, prev);
    LAUNCHED();
    lac::k_selz_compact<<<grid, 256, 0, st>>>(R, M5, npx, ws.zone, lists, list_words, prev);
    LAUNCHED();
    lac::k_selz_resolve<<<lac::SELZ_CLUSTER, lac::SELZ_RT, 0, st>>>(ws.sel, ws.zone, ws.histz, lists, list_words, rn2, gain_out,
                                                                    stats, prev);
    LAUNCHED();
    {
        // the selections by radix passes over the planes: one cooperative launch, which returns at once when the fast
        // path has done them.  Its grid must be resident as a whole.
        const int grid_c = std::min(grid, sms * std::max(1, std::min(di.occ_rounds, LAC_SEL_CTAS_PER_SM)));
        const uint32_t *zdone = &ws.zone->done, *zmdone = &ws.zone->mdone, *zno = &ws.zone->no;
        void* args[] = {(void*)&R, (void*)&M5, (void*)&npx, (void*)&ws.sel, (void*)&ws.hist, (void*)&rn2, (void*)&gain_out,
                        (void*)&stats, (void*)&prev, (void*)&zdone, (void*)&zmdone, (void*)&zno, (void*)&olist};
        CK(cudaLaunchCooperativeKernel((const void*)lac::k_sel_rounds, dim3((unsigned)grid_c), dim3(256), args, 0, st));
        LAUNCHED();
    }
    return LACOSMIC_OK;
}

__global__ void k_fill_floats(float* dst, int n, float v) {
    for (int i = threadIdx.x; i < n; i += blockDim.x) dst[i] = v;
}

int pack_bits(const uint8_t* mask_u8, uint32_t* bits, int h, int w, uint32_t* or_into, cudaStream_t st) {
    const unsigned nbx = (unsigned)((w + 255) / 256);
    lac::k_pack_bits<<<nbx * (unsigned)h, 256, 0, st>>>(mask_u8, bits, h, w, words_per_row(w), (int)nbx, or_into);
    LAUNCHED();
    return LACOSMIC_OK;
}

// R25: out = (med5(img) >= satlevel) dilated `grow` times (3x3); tmp: a second bit-plane
int satstar_bits(const float* img, int h, int w, float satlevel, int grow, uint32_t* out, uint32_t* tmp, cudaStream_t st) {
    const int wpr = words_per_row(w);
    const unsigned nbx = (unsigned)((w + 255) / 256), nbw = (unsigned)((wpr + 255) / 256);
    // the plane that ends up in `out` after `grow` ping-pong dilations
    uint32_t* a = (grow & 1) ? tmp : out;
    uint32_t* b = (grow & 1) ? out : tmp;
    lac::k_pack_ge<<<nbx * (unsigned)h, 256, 0, st>>>(img, satlevel, b, h, w, wpr, (int)nbx);
    LAUNCHED();
    lac::k_satcore<<<nbw * (unsigned)h, 256, 0, st>>>(b, a, h, w, wpr, (int)nbw);
    LAUNCHED();
    for (int j = 0; j < grow; ++j) {
        lac::k_dilate3<<<bit_grid(h, w), 256, 0, st>>>(a, b, h, w, wpr, bit_nbx(w));
        LAUNCHED();
        std::swap(a, b);
    }
    return LACOSMIC_OK;   // a == out
}

inline int check_variant(const lacosmic_variant* v) {
    if (!v) return LACOSMIC_OK;
    if (v->fsmode != LACOSMIC_FS_ADU && v->fsmode != LACOSMIC_FS_NORMALISED) return LACOSMIC_ERR_PARAM;
    if (v->satgrow < -1 || v->satgrow > LACOSMIC_MAX_SATGROW) return LACOSMIC_ERR_PARAM;
    if ((uintptr_t)v->var & 15) return LACOSMIC_ERR_ALIGN;
    return LACOSMIC_OK;
}

// A frame that is still arriving (lacosmic_run_host*): rows [0, row_end[b]) of img are on the device once ready[b] has
// fired.  The first noise/S pass is then launched band by band behind the copies instead of behind the whole frame.
constexpr int MAX_BANDS = LACOSMIC_HOST_BANDS;
static_assert(lac::NS_TH == LACOSMIC_HOST_TILE_ROWS && lac::NS_MY == LACOSMIC_HOST_TILE_MARGIN, "header and library disagree");
struct BandSync {
    int n = 0;
    cudaEvent_t ready[MAX_BANDS];
    int row_end[MAX_BANDS];
    int upto[MAX_BANDS];      // rows of tiles of the first pass that may run once band b has arrived (cumulative)
};

// The plan of the banded copy, a function of the shape alone (exported as lacosmic_host_band_plan so that a test can
// check the margin for every height without a GPU).  Band b ends at row row_end[b] (exclusive); once it has arrived,
// the rows of tiles below upto[b] may run.  A row of tiles j of the noise/S pass reads input rows
// [j * NS_TH - NS_MY, (j + 1) * NS_TH + NS_MY) (its TMA box, kernels.cuh), so it is released only when
// (j + 1) * NS_TH + NS_MY <= row_end[b], or when the band is the last one (the whole frame is there).
// Returns the number of bands; 0 = this shape is copied in one piece.
int band_plan(int h, int w, int* row_end, int* upto) {
    const int nty = (h + lac::NS_TH - 1) / lac::NS_TH;
    if ((w % 4) != 0 || nty < 4 * MAX_BANDS) return 0;
    int done = 0;
    for (int b = 0; b < MAX_BANDS; ++b) {
        const int re = b == MAX_BANDS - 1 ? h : std::min(h, (int)((long long)nty * (b + 1) / MAX_BANDS) * lac::NS_TH);
        int u = re >= h ? nty : (re - lac::NS_MY) / lac::NS_TH;      // rows of tiles wholly fed by rows < re
        u = std::max(done, std::min(u, nty));
        row_end[b] = re;
        upto[b] = u;
        done = u;
    }
    return MAX_BANDS;
}

// The iteration loop (O0-O7) for one frame.  vr: nullable variants (R22-R25).
int run_frame(const float* img, int h, int w, const lacosmic_params& p, uint8_t* mask_out,
              float* clean_out, const Workspace& ws, int32_t* iter_counts, const lacosmic_debug* dbg,
              cudaStream_t st, const lacosmic_variant* vr = nullptr, const BandSync* bands = nullptr) {
    const size_t P = (size_t)h * w;
    const int wpr = words_per_row(w);
    const size_t bp_bytes = (size_t)h * wpr * 4;
    float* work = clean_out;
    Span whole(KC_STEP, st);   // the whole frame, copies included
    const bool lazy = p.mode == LACOSMIC_MODE_LAZY;
    const float* var = vr ? vr->var : nullptr;                        // R24
    const bool fs1 = vr && vr->fsmode == LACOSMIC_FS_NORMALISED;      // R22
    const bool estimate = p.gain == 0.0f && !var;   // R21: no gain supplied (a variance plane replaces the noise model)
    // R23 / R25: the planes of the pixels never flagged / never donors, fixed for the frame
    const uint32_t *nok = nullptr, *donx = nullptr;
    if (vr && p.niter > 0 && (vr->bpm || vr->satgrow >= 0)) {
        int rc;
        if (vr->satgrow >= 0) {
            if ((rc = satstar_bits(img, h, w, p.satlevel, vr->satgrow, ws.NOK, ws.M2, st))) return rc;
        } else {
            CK(cudaMemsetAsync(ws.NOK, 0, bp_bytes, st));
        }
        if (vr->bpm) {
            if ((rc = pack_bits(vr->bpm, ws.DONX, h, w, ws.NOK, st))) return rc;
            donx = ws.DONX;
        }
        nok = ws.NOK;
    }
    // O0.  The lazy path fuses work = img_in into its first pass (which then reads img_in itself).
    const bool fused_copy = lazy && p.niter > 0;
    if (!fused_copy) CK(cudaMemcpyAsync(work, img, P * 4, cudaMemcpyDeviceToDevice, st));
    // Lazy frames whose first launch is the noise/S kernel itself: that pass clears the uint8 mask and k_grow_replace
    // sets the flagged pixels in it, which saves the bit-plane -> uint8 expansion (a launch and 29 MB) at the frame's end
    const bool direct_mask = fused_copy && mask_out && !estimate && !var && ((uintptr_t)mask_out & 3) == 0;
    // C = 0 and the counter block: cleared by the first kernels of the frame (k_list_candidates clears C in the
    // lazy path, the first noise pass clears the counters); plain memsets where those kernels do not run
    const bool fused_zero = p.niter > 0;
    if (!(lazy && p.niter > 0)) CK(cudaMemsetAsync(ws.C[0], 0, bp_bytes, st));
    if (!fused_zero) CK(cudaMemsetAsync((char*)ws.S + ws.zero_off, 0, ws.zero_bytes, st));
    int* const zero_ptr = (int*)((char*)ws.S + ws.zero_off);
    const int zero_n = (int)(ws.zero_bytes / 4);
    const float siglow = p.sigfrac * p.sigclip;   // R9: one fp32 multiply on the host
    const float rn2 = p.readnoise * p.readnoise;
    lac::GateParams gp{p.sigclip, siglow, p.objlim, p.satlevel};
    dim3 tb(lac::NT);
    const int tgx = (w + lac::TW - 1) / lac::TW, tgy = (h + lac::TH - 1) / lac::TH;
    // TMA path needs 16-byte row pitch; other widths take the generic tile loader
    const bool tma = (w % 4 == 0);
    const int ntx = tgx, ntiles = tgx * tgy;
    const int ntilesNS = ntx * ((h + lac::NS_TH - 1) / lac::NS_TH);   // tiles of the noise/S pass
    CUtensorMap mapWorkNS, mapImgNS, mapWorkFG, mapS;
    int gridNS = 0, gridFG = 0, gridQ = 1184, gridE = 2368;
    if (p.niter > 0) {
        const DeviceInfo& di = device_info();
        if (!di.ok) { g_last_cuda_error = (int)cudaGetLastError(); return LACOSMIC_ERR_CUDA; }
        gridQ = di.sms * di.occ_quads;
        gridE = di.sms * di.occ_eval;
        if (tma) {
            if (!make_map(&mapWorkNS, work, h, w, lac::NS_PITCH, lac::NS_ROWS) ||
                !make_map(&mapImgNS, img, h, w, lac::NS_PITCH, lac::NS_ROWS) ||
                !make_map(&mapWorkFG, work, h, w, lac::FG_PA, lac::FG_AROWS) ||
                !make_map(&mapS, ws.S, h, w, lac::FG_PS, lac::FG_SROWS)) {
                g_last_cuda_error = (int)cudaErrorInvalidValue;
                return LACOSMIC_ERR_CUDA;
            }
            // several CTAs per resident slot: the hardware hands a slot the next CTA as soon as one retires, which
            // balances the tail (measured on B200, configs[2]: 0.204 ms with one CTA per slot, 0.193 with six; one tile
            // per CTA, i.e. no prefetch across tiles, 0.200)
            gridNS = std::min(ntilesNS, di.sms * di.occ_noise * LAC_NS_WAVES);
            gridFG = std::min(ntiles, di.sms * di.occ_fine * LAC_FG_WAVES);
        }
    }
    for (int t = 0; t < p.niter; ++t) {
        const int* prev = t > 0 ? ws.counts + (t - 1) : nullptr;
        const bool d = dbg && dbg->iter == t;
        int rc = LACOSMIC_OK;
        const float* src = (fused_copy && t == 0) ? img : work;
        // tiles tile0 .. tile0 + nt - 1 of the noise/S pass (TMA path; the generic path always runs the whole frame)
        auto noise_tiles = [&](const lac::NoiseArgs& na, const float* from, int tile0, int nt) -> int {
            const CUtensorMap& map = from == img ? mapImgNS : mapWorkNS;
            const int g = std::min(nt, gridNS);
            // the configurations of a plain frame are compiled without the tests of the nullable outputs
            const bool plain = !na.dbgLp && !na.dbgN && !na.R && !na.gain_dev;
            const bool resid = na.R && !na.dbgLp && !na.dbgN && !na.gain_dev && !na.A1 && !na.mask_zero && !na.var;
            if (plain && na.copy_out && na.A1 && na.mask_zero) launch_pdl(lac::k_noise_S_tma<7>, dim3(g), tb, lac::NS_SMEM_BYTES, st, map, na, ntx, nt, prev, tile0);
            else if (plain && na.copy_out && na.A1 && !na.mask_zero) launch_pdl(lac::k_noise_S_tma<3>, dim3(g), tb, lac::NS_SMEM_BYTES, st, map, na, ntx, nt, prev, tile0);
            else if (plain && !na.copy_out && !na.A1 && !na.mask_zero) launch_pdl(lac::k_noise_S_tma<0>, dim3(g), tb, lac::NS_SMEM_BYTES, st, map, na, ntx, nt, prev, tile0);
            else if (resid && na.copy_out) launch_pdl(lac::k_noise_S_tma<9>, dim3(g), tb, lac::NS_SMEM_BYTES, st, map, na, ntx, nt, prev, tile0);
            else if (resid && !na.copy_out) launch_pdl(lac::k_noise_S_tma<8>, dim3(g), tb, lac::NS_SMEM_BYTES, st, map, na, ntx, nt, prev, tile0);
            else launch_pdl(lac::k_noise_S_tma<-1>, dim3(g), tb, lac::NS_SMEM_BYTES, st, map, na, ntx, nt, prev, tile0);
            LAUNCHED();
            return LACOSMIC_OK;
        };
        auto noise_pass = [&](const lac::NoiseArgs& na, const float* from) -> int {
            Span sp(KC_NOISE_S, st);
            if (!tma) {
                lac::k_noise_S<<<ntilesNS, tb, 0, st>>>(from, na, ntx, prev);
                LAUNCHED();
                return LACOSMIC_OK;
            }
            if (bands && t == 0 && from == img && bands->n > 0) {
                // the frame is still arriving: a row of tiles (NS_TH rows + 2 rows of margin below) runs as soon as the
                // band that holds its last input row is on the device
                const int ntyNS = ntilesNS / ntx;
                int done = 0;                          // rows of tiles launched so far
                for (int b = 0; b < bands->n; ++b) {
                    CK(cudaStreamWaitEvent(st, bands->ready[b], 0));
                    const int upto = bands->upto[b];                                 // band_plan: rows of tiles wholly fed by now
                    if (upto > done) {
                        int rc2 = noise_tiles(na, from, done * ntx, (upto - done) * ntx);
                        if (rc2) return rc2;
                        done = upto;
                    }
                }
                if (done < ntyNS) return noise_tiles(na, from, done * ntx, (ntyNS - done) * ntx);
                return LACOSMIC_OK;
            }
            return noise_tiles(na, from, 0, ntilesNS);
        };
        if (estimate) {
            // R21: the gain of this iteration from its input image.  One dense pass writes the residual plane
            // (into the candidate list's storage, which is not in use yet), med5(work) into the S plane and, at
            // t = 0, the work = img_in copy.  The selection leaves the gain in ws.gains[t].
            lac::NoiseArgs ne{ws.S, nullptr, nullptr, nullptr, nullptr, (fused_copy && t == 0) ? work : nullptr,
                              h, w, wpr, 1.0f, rn2, p.sigclip, siglow, p.satlevel, (float*)ws.clist, nullptr,
                              t == 0 ? zero_ptr : nullptr, zero_n};
            if ((rc = noise_pass(ne, src))) return rc;
            if ((rc = sigma_clip_gain((const float*)ws.clist, ws.S, P, ws, ws.qlist, (size_t)((char*)ws.C[0] - (char*)ws.qlist) / 4, rn2, ws.gains + t, nullptr, prev, st))) return rc;
            src = work;
        }
        // lazy path, t >= 1: S, A1, A2 and the tests only change near the pixels the previous replacement
        // rewrote (ws.NEED); a debug dump recomputes the planes everywhere, and so does an estimated gain
        // (it changes with every iteration, and S with it)
        const bool incr = lazy && t > 0 && !d && !estimate;
        // R22 in the dense path: the gate kernel reads the noise plane, which the noise/S pass stores in the
        // candidate list's storage (not used by the dense path; free again once a gain estimate has been selected)
        float* const nplane = (d && dbg->N) ? dbg->N : ((fs1 && !lazy) ? (float*)ws.clist : nullptr);
        lac::NoiseArgs na{ws.S, d ? dbg->Lp : nullptr, nplane,
                          lazy ? ws.A1 : nullptr, lazy ? ws.A2 : nullptr,
                          (fused_copy && t == 0 && !estimate) ? work : nullptr,
                          h, w, wpr, p.gain, rn2, p.sigclip, siglow, p.satlevel, nullptr,
                          estimate ? ws.gains + t : nullptr, (t == 0 && !estimate) ? zero_ptr : nullptr, zero_n,
                          nok, var, (direct_mask && t == 0) ? mask_out : nullptr};
        if (incr) {
            {
                Span sp(KC_LISTS, st);
                launch_pdl(lac::k_dirty_lists, dim3(grow_grid(h, w)), dim3(32 * lac::WG_WARPS), 0, st, ws.NEED, ws.A1, ws.G1, ws.G2, ws.G2F,
                           ws.M1, ws.qlist, ws.nquad + t, ws.clist, ws.ncand + t, h, w, wpr, grow_nbx(w), prev);
                LAUNCHED();
            }
            {
                Span sp(KC_NOISE_S_QUADS, st);
                launch_pdl(lac::k_noise_S_quads, dim3(gridQ), dim3(256), 0, st, work, na, ws.qlist, ws.nquad + t, ws.clist, ws.ncand + t, prev);
                LAUNCHED();
            }
        } else {
            if (estimate || var) {
                // the residual pass left med5(work) in the S plane (R21), or N comes from the variance plane (R24):
                // S, A1, A2 follow elementwise (HBM bound)
                Span sp(KC_NOISE_S, st);
                const unsigned nbx = (unsigned)((w + 127) / 128);
                if (tma) lac::k_S_from_m5<<<nbx * (unsigned)((h + 8 * lac::SM5_ROWS - 1) / (8 * lac::SM5_ROWS)), 256, 0, st>>>(src, na, (int)nbx, prev);
                else lac::k_S_from_m5_generic<<<nbx * (unsigned)((h + 7) / 8), 256, 0, st>>>(src, na, (int)nbx, prev);
                LAUNCHED();
            } else if ((rc = noise_pass(na, src))) {
                return rc;
            }
            if (lazy) {
                Span sp(KC_LISTS, st);
                launch_pdl(lac::k_list_candidates, dim3(bit_grid(h, w)), dim3(256), 0, st, ws.A1, (t > 0 && !estimate) ? ws.NEED : nullptr,
                           ws.G1, ws.G2, ws.G2F, ws.M1, ws.clist, ws.ncand + t, t == 0 ? ws.C[0] : nullptr, h, w, wpr, bit_nbx(w), prev);
                LAUNCHED();
            }
        }
        if (lazy) {
            // steps (3b)-(5) on the listed candidates only (lazy.cuh)
            lac::CandArgs ca{ws.S, work, ws.G1, ws.G2, ws.M1, h, w, wpr, p.sigclip, siglow, p.objlim,
                             p.gain, rn2, estimate ? ws.gains + t : nullptr, var, g_stats ? ws.nfine + t : nullptr};
            Span sp(KC_EVAL, st);
            if (fs1) launch_pdl(lac::k_eval_candidates<1>, dim3(gridE), dim3(128), 0, st, ca, ws.clist, ws.ncand + t, prev);
            else launch_pdl(lac::k_eval_candidates<0>, dim3(gridE), dim3(128), 0, st, ca, ws.clist, ws.ncand + t, prev);
            LAUNCHED();
        } else {
            lac::FineArgs fa{ws.G1, ws.G2, ws.M1, d ? dbg->Sp : nullptr, d ? dbg->m3 : nullptr,
                             d ? dbg->F : nullptr, h, w, wpr, gp, fs1 ? nplane : nullptr, nok};
            Span sp(KC_FINE_GATES, st);
            if (tma) lac::k_fine_gates_tma<<<gridFG, tb, lac::FG_SMEM_BYTES, st>>>(mapWorkFG, mapS, fa, ntx, ntiles, prev);
            else lac::k_fine_gates<<<(unsigned)ntiles, tb, 0, st>>>(work, ws.S, fa, ntx, prev);
            LAUNCHED();
        }
        if (d && dbg->S) CK(cudaMemcpyAsync(dbg->S, ws.S, P * 4, cudaMemcpyDeviceToDevice, st));
        // steps (6)-(7), fused; in the lazy path G2 is completed on the pixels the second growth reaches
        lac::GrowArgs ga{ws.M1, ws.G1, ws.G2, ws.G2F, lazy ? ws.A1 : nullptr, lazy ? ws.A2 : nullptr,
                         ws.C[t & 1], ws.C[(t + 1) & 1], ws.NEED, d ? ws.M2 : nullptr, d ? ws.M3 : nullptr,
                         ws.S, img, work, ws.counts + t, incr ? 1 : 0, h, w, wpr, siglow, grow_nbx(w),
                         donx, g_stats ? ws.nneed + t : nullptr, direct_mask ? mask_out : nullptr};
        if ((rc = grow_replace(ga, prev, st))) return rc;
        if (d) {
            // lazy path: G2 is only evaluated where step (6) needs it, so it is not dumped
            struct { const uint32_t* b; uint8_t* o; } planes[] = {
                {ws.G1, dbg->G1}, {ws.G2, lazy ? nullptr : dbg->G2}, {ws.M1, dbg->M1},
                {ws.M2, dbg->M2}, {ws.M3, dbg->M3}, {ws.C[(t + 1) & 1], dbg->C}};
            for (auto& pl : planes)
                if (pl.o && (rc = unpack(pl.b, pl.o, h, w, st))) return rc;
        }
    }
    const bool want_counts = iter_counts && p.niter > 0;
    // mask_out null: the caller reads the bit-plane.  The iteration counts ride along with the unpack launch.
    int rc = (mask_out && !direct_mask)
                 ? unpack(ws.C[p.niter & 1], mask_out, h, w, st, ws.counts, want_counts ? iter_counts : nullptr, p.niter)
                 : LACOSMIC_OK;
    if (rc) return rc;
    if (want_counts && (!mask_out || direct_mask))
        CK(cudaMemcpyAsync(iter_counts, ws.counts, (size_t)p.niter * 4, cudaMemcpyDeviceToDevice, st));
    if (dbg && dbg->gains && p.niter > 0) {
        if (!estimate) {
            k_fill_floats<<<1, 64, 0, st>>>(ws.gains, p.niter, p.gain);
            LAUNCHED();
        }
        CK(cudaMemcpyAsync(dbg->gains, ws.gains, (size_t)p.niter * 4, cudaMemcpyDeviceToDevice, st));
    }
    return LACOSMIC_OK;
}

// R26 (comparison only): out = sepmedK(in), tmp = the row pass
int sepmed(const float* in, float* out, float* tmp, int h, int w, int k, cudaStream_t st) {
    const unsigned g = (unsigned)(((size_t)h * w + 255) / 256);
    if (k == 3) { lac::k_sepmed_pass<3, true><<<g, 256, 0, st>>>(in, tmp, h, w); lac::k_sepmed_pass<3, false><<<g, 256, 0, st>>>(tmp, out, h, w); }
    else if (k == 5) { lac::k_sepmed_pass<5, true><<<g, 256, 0, st>>>(in, tmp, h, w); lac::k_sepmed_pass<5, false><<<g, 256, 0, st>>>(tmp, out, h, w); }
    else { lac::k_sepmed_pass<7, true><<<g, 256, 0, st>>>(in, tmp, h, w); lac::k_sepmed_pass<7, false><<<g, 256, 0, st>>>(tmp, out, h, w); }
    g_launches += 1;
    LAUNCHED();
    return LACOSMIC_OK;
}

// O0-O7 with every median replaced by the separable one (R26).  Planes: A = ws.S, B = the candidate list's storage,
// C3 = `third` (the extra plane of lacosmic_sepmed_workspace_bytes).
int run_sepmed_frame(const float* img, int h, int w, const lacosmic_params& p, uint8_t* mask_out, float* clean_out,
                     const Workspace& ws, float* third, int32_t* iter_counts, const lacosmic_debug* dbg, cudaStream_t st) {
    const size_t P = (size_t)h * w;
    const int wpr = words_per_row(w);
    const size_t bp_bytes = (size_t)h * wpr * 4;
    float *work = clean_out, *A = ws.S, *B = (float*)ws.clist, *C3 = third;
    CK(cudaMemcpyAsync(work, img, P * 4, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemsetAsync(ws.C[0], 0, bp_bytes, st));
    CK(cudaMemsetAsync((char*)ws.S + ws.zero_off, 0, ws.zero_bytes, st));
    const float siglow = p.sigfrac * p.sigclip, rn2 = p.readnoise * p.readnoise;
    const unsigned gw = (unsigned)(((size_t)h * wpr + 7) / 8);
    for (int t = 0; t < p.niter; ++t) {
        const int* prev = t > 0 ? ws.counts + (t - 1) : nullptr;
        const bool d = dbg && dbg->iter == t;
        int rc;
        // O2, O3a: A = sepmed5(work), then S in place (with L+ and N)
        if ((rc = sepmed(work, A, B, h, w, 5, st))) return rc;
        lac::NoiseArgs na{A, d ? dbg->Lp : nullptr, d ? dbg->N : nullptr, nullptr, nullptr, nullptr, h, w, wpr,
                          p.gain, rn2, p.sigclip, siglow, p.satlevel, nullptr, nullptr, nullptr, 0};
        const unsigned nbx = (unsigned)((w + 127) / 128);
        lac::k_S_from_m5_generic<<<nbx * (unsigned)((h + 7) / 8), 256, 0, st>>>(work, na, (int)nbx, nullptr);
        LAUNCHED();
        if (d && dbg->S) CK(cudaMemcpyAsync(dbg->S, A, P * 4, cudaMemcpyDeviceToDevice, st));
        // O3b, O5: C3 = sepmed5(S); G1, G2
        if ((rc = sepmed(A, C3, B, h, w, 5, st))) return rc;
        lac::SepGateArgs ga{work, A, C3, nullptr, nullptr, ws.G1, ws.G2, ws.M1, d ? dbg->Sp : nullptr, d ? dbg->F : nullptr,
                            h, w, wpr, p.sigclip, siglow, p.objlim, p.satlevel};
        lac::k_sep_gates<0><<<gw, 256, 0, st>>>(ga);
        LAUNCHED();
        // O4, O5: A = m3 = sepmed3(work); C3 = sepmed7(m3); M1
        if ((rc = sepmed(work, A, B, h, w, 3, st))) return rc;
        if (d && dbg->m3) CK(cudaMemcpyAsync(dbg->m3, A, P * 4, cudaMemcpyDeviceToDevice, st));
        if ((rc = sepmed(A, C3, B, h, w, 7, st))) return rc;
        ga.m3 = A;
        ga.m7 = C3;
        lac::k_sep_gates<1><<<gw, 256, 0, st>>>(ga);
        LAUNCHED();
        // O6, O7: the product kernel (G2 complete, as in the dense path)
        lac::GrowArgs gr{ws.M1, ws.G1, ws.G2, ws.G2F, nullptr, nullptr, ws.C[t & 1], ws.C[(t + 1) & 1], ws.NEED,
                         d ? ws.M2 : nullptr, d ? ws.M3 : nullptr, A, img, work, ws.counts + t, 0, h, w, wpr, siglow,
                         grow_nbx(w), nullptr, nullptr, nullptr};
        if ((rc = grow_replace(gr, prev, st))) return rc;
        if (d) {
            struct { const uint32_t* b; uint8_t* o; } planes[] = {{ws.G1, dbg->G1}, {ws.G2, dbg->G2}, {ws.M1, dbg->M1},
                                                                 {ws.M2, dbg->M2}, {ws.M3, dbg->M3}, {ws.C[(t + 1) & 1], dbg->C}};
            for (auto& pl : planes)
                if (pl.o && (rc = unpack(pl.b, pl.o, h, w, st))) return rc;
        }
    }
    const bool want_counts = iter_counts && p.niter > 0;
    return unpack(ws.C[p.niter & 1], mask_out, h, w, st, ws.counts, want_counts ? iter_counts : nullptr, p.niter);
}

// Internal streams of lacosmic_run_batch (per calling thread and device, created on first use, kept for the
// life of the thread): non-blocking, forked from / joined into the caller's stream with events.
struct BatchStreams {
    int dev = -1;
    cudaStream_t st[LACOSMIC_MAX_BATCH_STREAMS];
    cudaEvent_t fork, join[LACOSMIC_MAX_BATCH_STREAMS];
    cudaStream_t copy;                  // H2D copies of a single host frame, band by band (run_host_frame)
    cudaEvent_t band[MAX_BANDS];
};
BatchStreams* batch_streams() {
    thread_local BatchStreams pool[16];
    thread_local int npool = 0;
    int dev = 0;
    if (!cuda_ok(cudaGetDevice(&dev))) return nullptr;
    for (int i = 0; i < npool; ++i)
        if (pool[i].dev == dev) return &pool[i];
    if (npool == 16) return nullptr;
    BatchStreams& b = pool[npool];
    if (!cuda_ok(cudaEventCreateWithFlags(&b.fork, cudaEventDisableTiming))) return nullptr;
    for (int s = 0; s < LACOSMIC_MAX_BATCH_STREAMS; ++s) {
        if (!cuda_ok(cudaStreamCreateWithFlags(&b.st[s], cudaStreamNonBlocking))) return nullptr;
        if (!cuda_ok(cudaEventCreateWithFlags(&b.join[s], cudaEventDisableTiming))) return nullptr;
    }
    if (!cuda_ok(cudaStreamCreateWithFlags(&b.copy, cudaStreamNonBlocking))) return nullptr;
    for (int k = 0; k < MAX_BANDS; ++k)
        if (!cuda_ok(cudaEventCreateWithFlags(&b.band[k], cudaEventDisableTiming))) return nullptr;
    b.dev = dev;
    ++npool;
    return &b;
}

int check_frame_args(const float* img, int h, int w, const lacosmic_params* p, const uint8_t* mask_out,
                     const float* clean_out, const void* workspace, size_t workspace_bytes) {
    if (!img || !p || !mask_out || !clean_out || !workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((rc = check_params(*p))) return rc;
    if (((uintptr_t)img & 15) || ((uintptr_t)clean_out & 15) || ((uintptr_t)workspace & 255))
        return LACOSMIC_ERR_ALIGN;
    size_t P = (size_t)h * w, need = lacosmic_workspace_bytes(h, w);
    if (workspace_bytes < need) return LACOSMIC_ERR_WORKSPACE;
    if (overlap(img, P * 4, clean_out, P * 4) || overlap(img, P * 4, mask_out, P) ||
        overlap(clean_out, P * 4, mask_out, P) || overlap(workspace, need, img, P * 4) ||
        overlap(workspace, need, clean_out, P * 4) || overlap(workspace, need, mask_out, P))
        return LACOSMIC_ERR_ALIAS;
    return LACOSMIC_OK;
}

}  // namespace

extern "C" {

size_t lacosmic_workspace_bytes(int h, int w) {
    if (check_shape(h, w)) return 0;
    return carve(nullptr, h, w).bytes;
}

extern "C++" {
namespace {
// ---- replay of a repeated frame call from a CUDA graph ------------------------------------------
// The launch sequence of a frame is a pure function of the call's arguments (pointers, shape, parameters): what
// the kernels do with the data is decided on the device.  A pipeline that cleans frame after frame through the
// same buffers therefore enqueues the same 16 launches every time; from the second identical call on, the
// sequence is captured once into a CUDA graph and later calls replay it (one graph launch instead of 16 kernel
// launches: ~2 us less launch latency per dependent kernel, 0.03 ms per 4000x6500 frame on B200).  Every kernel
// still runs on every call -- only the host-side launch work is reused.  Not used with a debug dump, with kernel
// timing or statistics on, on the legacy default stream or on a stream that is being captured by the caller.
struct GraphKey {
    int dev, h, w;
    int gain_fast;            // which path of the gain estimate the captured sequence takes (a process-wide switch)
    const void *img, *mask, *clean, *ws, *counts;
    size_t ws_bytes;
    lacosmic_params p;
    bool operator==(const GraphKey& o) const {
        return dev == o.dev && h == o.h && w == o.w && gain_fast == o.gain_fast && img == o.img && mask == o.mask &&
               clean == o.clean && ws == o.ws && counts == o.counts && ws_bytes == o.ws_bytes &&
               std::memcmp(&p, &o.p, sizeof p) == 0;
    }
};
// Locking.  g_graph_mu guards the table itself (keys, seen / used / users / doomed) and is held only for the look-up
// and the release, never across a CUDA call that takes long.  An entry's own `mu` is held while its graph is
// captured, instantiated and launched (a cudaGraphExec_t must not be launched from two threads at once), so threads
// that work with different argument sets -- different GPUs, streams, frames -- do not wait for each other.  An entry
// with users > 0 is neither evicted nor destroyed; lacosmic_graph_replay_enable(0) marks it doomed and its last user
// destroys it.
struct GraphEntry {
    GraphKey key;
    cudaGraphExec_t exec = nullptr;
    int launches = 0;
    int seen = 0;             // calls with this key so far
    bool failed = false;      // capture or instantiation failed once: this key always takes the direct path
    bool doomed = false;      // the replay was switched off while a thread was using the entry
    int users = 0;            // threads between look-up and release
    unsigned long long used = 0;
    std::mutex mu;
    void reset() {            // g_graph_mu held, users == 0
        if (exec) cudaGraphExecDestroy(exec);
        exec = nullptr;
        launches = seen = 0;
        failed = doomed = false;
        used = 0;
    }
};
constexpr int GRAPH_CACHE = 16;
GraphEntry g_graphs[GRAPH_CACHE];
std::mutex g_graph_mu;
unsigned long long g_graph_clock = 0;
int g_graphs_on = -1;         // -1: not decided yet (environment LACOSMIC_GRAPHS=0 switches the replay off); under g_graph_mu

bool graphs_enabled() {
    if (g_graphs_on < 0) {
        const char* e = std::getenv("LACOSMIC_GRAPHS");
        g_graphs_on = (e && e[0] == '0') ? 0 : 1;
    }
    return g_graphs_on == 1;
}
}  // namespace
}

int lacosmic_graph_replay_enable(int enable) {
    std::lock_guard<std::mutex> lock(g_graph_mu);
    g_graphs_on = enable ? 1 : 0;
    if (!enable)
        for (GraphEntry& e : g_graphs) {
            if (e.users > 0) e.doomed = true;
            else e.reset();
        }
    return LACOSMIC_OK;
}

int lacosmic_run_ws(const float* img, int h, int w, const lacosmic_params* p, uint8_t* mask_out,
                    float* clean_out, void* workspace, size_t workspace_bytes, int32_t* iter_counts,
                    const lacosmic_debug* dbg, void* stream) {
    g_launches = 0;
    int rc = check_frame_args(img, h, w, p, mask_out, clean_out, workspace, workspace_bytes);
    if (rc) return rc;
    if (dbg && (dbg->iter < -1 || dbg->iter >= LACOSMIC_MAX_NITER)) return LACOSMIC_ERR_PARAM;
    if (dbg)   // fp32 debug planes are written with 16-byte vectors
        for (const float* pl : {dbg->Lp, dbg->N, dbg->S, dbg->Sp, dbg->m3, dbg->F})
            if ((uintptr_t)pl & 15) return LACOSMIC_ERR_ALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    const Workspace ws = carve(workspace, h, w);
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    const bool replayable = !dbg && !g_kt.enabled && !g_stats && p->niter > 0 && st != nullptr && st != cudaStreamLegacy &&
                            cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap == cudaStreamCaptureStatusNone;
    if (!replayable) {
        cudaGetLastError();     // cudaStreamIsCapturing on the legacy stream during someone else's capture reports an error
        return run_frame(img, h, w, *p, mask_out, clean_out, ws, iter_counts, dbg, st);
    }
    GraphKey key;
    std::memset(&key, 0, sizeof key);
    cudaGetDevice(&key.dev);
    key.h = h; key.w = w; key.img = img; key.mask = mask_out; key.clean = clean_out; key.ws = workspace;
    key.counts = iter_counts; key.ws_bytes = workspace_bytes; key.p = *p;
    key.gain_fast = gain_fast_enabled() ? 1 : 0;
    GraphEntry* e = nullptr;
    {   // look-up: the only part under the table lock
        std::lock_guard<std::mutex> lock(g_graph_mu);
        if (graphs_enabled()) {
            GraphEntry* lru = nullptr;
            for (GraphEntry& g : g_graphs) {
                if (g.seen && !g.doomed && g.key == key) { e = &g; break; }
                if (g.users == 0 && (!lru || g.used < lru->used)) lru = &g;
            }
            if (e) {
                e->used = ++g_graph_clock;
                ++e->seen;
                ++e->users;
            } else if (lru) {       // first call with these arguments: remember them, run directly
                lru->reset();
                lru->key = key;
                lru->seen = 1;
                lru->used = ++g_graph_clock;
            }                       // (every entry in use by another thread: run directly, remember nothing)
        }
    }
    if (!e) return run_frame(img, h, w, *p, mask_out, clean_out, ws, iter_counts, dbg, st);
    bool launched = false, launch_failed = false;
    {
        std::lock_guard<std::mutex> mine(e->mu);
        if (!e->exec && !e->failed) {   // second call: capture the sequence
            cudaGraph_t graph = nullptr;
            if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                rc = run_frame(img, h, w, *p, mask_out, clean_out, ws, iter_counts, dbg, st);
                const cudaError_t ce = cudaStreamEndCapture(st, &graph);
                if (rc == LACOSMIC_OK && ce == cudaSuccess && graph &&
                    cudaGraphInstantiate(&e->exec, graph, 0) == cudaSuccess) {
                    e->launches = g_launches;
                } else {
                    e->exec = nullptr;
                    e->failed = true;
                }
                if (graph) cudaGraphDestroy(graph);
            } else {
                e->failed = true;
            }
            cudaGetLastError();
        }
        if (e->exec) {
            g_launches = e->launches;
            launched = true;
            launch_failed = !cuda_ok(cudaGraphLaunch(e->exec, st));
        }
    }
    {   // release
        std::lock_guard<std::mutex> lock(g_graph_mu);
        if (--e->users == 0 && e->doomed) e->reset();
    }
    if (launched) return launch_failed ? LACOSMIC_ERR_CUDA : LACOSMIC_OK;
    g_launches = 0;
    return run_frame(img, h, w, *p, mask_out, clean_out, ws, iter_counts, dbg, st);
}

int lacosmic_run_ex(const float* img, int h, int w, const lacosmic_params* p, const lacosmic_variant* v,
                    uint8_t* mask_out, float* clean_out, void* workspace, size_t workspace_bytes,
                    int32_t* iter_counts, const lacosmic_debug* dbg, void* stream) {
    g_launches = 0;
    int rc = check_frame_args(img, h, w, p, mask_out, clean_out, workspace, workspace_bytes);
    if (rc) return rc;
    if ((rc = check_variant(v))) return rc;
    if (dbg && (dbg->iter < -1 || dbg->iter >= LACOSMIC_MAX_NITER)) return LACOSMIC_ERR_PARAM;
    if (dbg)
        for (const float* pl : {dbg->Lp, dbg->N, dbg->S, dbg->Sp, dbg->m3, dbg->F})
            if ((uintptr_t)pl & 15) return LACOSMIC_ERR_ALIGN;
    const size_t P = (size_t)h * w, need = lacosmic_workspace_bytes(h, w);
    // bpm / var are inputs read throughout the frame: they may coincide with nothing the frame writes (the outputs and
    // the workspace, whose first launches already write planes and counters).  They may alias img: all three are read-only.
    if (v && ((v->bpm && (overlap(v->bpm, P, clean_out, P * 4) || overlap(v->bpm, P, mask_out, P) ||
                          overlap(v->bpm, P, workspace, need))) ||
              (v->var && (overlap(v->var, P * 4, clean_out, P * 4) || overlap(v->var, P * 4, mask_out, P) ||
                          overlap(v->var, P * 4, workspace, need)))))
        return LACOSMIC_ERR_ALIAS;
    return run_frame(img, h, w, *p, mask_out, clean_out, carve(workspace, h, w), iter_counts, dbg,
                     (cudaStream_t)stream, v);
}

int lacosmic_run(const float* img, int h, int w, float gain, float readnoise, float sigclip,
                 float sigfrac, float objlim, int niter, float satlevel, uint8_t* mask_out,
                 float* clean_out, void* stream) {
    g_launches = 0;
    lacosmic_params p{gain, readnoise, sigclip, sigfrac, objlim, satlevel, niter, LACOSMIC_MODE_LAZY};
    if (!img || !mask_out || !clean_out) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((rc = check_params(p))) return rc;
    size_t need = lacosmic_workspace_bytes(h, w);
    void* ws = nullptr;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMallocAsync(&ws, need, st));
    rc = check_frame_args(img, h, w, &p, mask_out, clean_out, ws, need);
    if (!rc) rc = run_frame(img, h, w, p, mask_out, clean_out, carve(ws, h, w), nullptr, nullptr, st);
    if (!cuda_ok(cudaFreeAsync(ws, st)) && !rc) rc = LACOSMIC_ERR_CUDA;
    return rc;
}

size_t lacosmic_batch_workspace_bytes(int h, int w, int concurrency) {
    if (check_shape(h, w) || concurrency < 1) return 0;
    return (size_t)std::min(concurrency, LACOSMIC_MAX_BATCH_STREAMS) * align_up(lacosmic_workspace_bytes(h, w), 256);
}

int lacosmic_run_batch(const float* imgs, int n, int h, int w, const lacosmic_params* params,
                       uint8_t* masks_out, float* cleans_out, void* workspace, size_t workspace_bytes,
                       int32_t* iter_counts, void* stream) {
    g_launches = 0;
    if (n < 0) return LACOSMIC_ERR_SHAPE;
    if (n == 0) return LACOSMIC_OK;
    if (!imgs || !params || !masks_out || !cleans_out || !workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    size_t P = (size_t)h * w;
    if ((P * 4) & 15) {
        // frames inside the batch must each stay 16-byte aligned
        if (n > 1) return LACOSMIC_ERR_ALIGN;
    }
    for (int f = 0; f < n; ++f) {
        rc = check_frame_args(imgs + f * P, h, w, params + f, masks_out + f * P, cleans_out + f * P,
                              workspace, workspace_bytes);
        if (rc) return rc;
    }
    if (overlap(imgs, n * P * 4, cleans_out, n * P * 4) || overlap(imgs, n * P * 4, masks_out, n * P) ||
        overlap(cleans_out, n * P * 4, masks_out, n * P))
        return LACOSMIC_ERR_ALIAS;
    const size_t slice = align_up(lacosmic_workspace_bytes(h, w), 256);
    const int k = (int)std::min<size_t>(std::min(n, LACOSMIC_MAX_BATCH_STREAMS), workspace_bytes / slice);
    if (overlap(workspace, (size_t)k * slice, imgs, n * P * 4) || overlap(workspace, (size_t)k * slice, cleans_out, n * P * 4) ||
        overlap(workspace, (size_t)k * slice, masks_out, n * P))
        return LACOSMIC_ERR_ALIAS;
    cudaStream_t caller = (cudaStream_t)stream;
    BatchStreams* bs = nullptr;
    if (k > 1) {
        bs = batch_streams();
        if (!bs) return LACOSMIC_ERR_CUDA;
        CK(cudaEventRecord(bs->fork, caller));
        for (int s = 0; s < k; ++s) CK(cudaStreamWaitEvent(bs->st[s], bs->fork, 0));
    }
    for (int f = 0; f < n; ++f) {
        const int s = f % k;
        cudaStream_t st = k > 1 ? bs->st[s] : caller;
        Workspace ws = carve((char*)workspace + (size_t)s * slice, h, w);
        rc = run_frame(imgs + f * P, h, w, params[f], masks_out + f * P, cleans_out + f * P, ws, nullptr,
                       nullptr, st);
        if (rc) break;
        if (iter_counts && !cuda_ok(cudaMemcpyAsync(iter_counts + (size_t)f * LACOSMIC_MAX_NITER, ws.counts,
                                                    LACOSMIC_MAX_NITER * 4, cudaMemcpyDeviceToDevice, st))) {
            rc = LACOSMIC_ERR_CUDA;
            break;
        }
    }
    if (k > 1) {   // join, also after an error: the caller's stream must not run ahead of work already enqueued
        for (int s = 0; s < k; ++s) {
            if (!cuda_ok(cudaEventRecord(bs->join[s], bs->st[s])) ||
                !cuda_ok(cudaStreamWaitEvent(caller, bs->join[s], 0)))
                rc = rc ? rc : LACOSMIC_ERR_CUDA;
        }
    }
    return rc;
}

size_t lacosmic_host_workspace_bytes(int h, int w) {
    if (check_shape(h, w)) return 0;
    size_t P = (size_t)h * w;
    return align_up(P * 4, 256) * 2 + align_up(P, 256) + lacosmic_workspace_bytes(h, w);
}

extern "C++" {
namespace {
// uint16 -> fp32 (exact), 8 pixels per thread; src and dst must not overlap
__global__ void __launch_bounds__(256) k_u16_to_f32(const uint16_t* __restrict__ src, float* __restrict__ dst, size_t n) {
    const size_t i = ((size_t)blockIdx.x * 256 + threadIdx.x) * 8;
    if (i + 8 <= n) {
        const uint4 q = __ldg(reinterpret_cast<const uint4*>(src + i));
        const uint32_t v[4] = {q.x, q.y, q.z, q.w};
        float o[8];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            o[2 * k] = (float)(v[k] & 0xffffu);
            o[2 * k + 1] = (float)(v[k] >> 16);
        }
        *reinterpret_cast<float4*>(dst + i) = make_float4(o[0], o[1], o[2], o[3]);
        *reinterpret_cast<float4*>(dst + i + 4) = make_float4(o[4], o[5], o[6], o[7]);
    } else {
        for (size_t k = i; k < n; ++k) dst[k] = (float)src[k];
    }
}

// Host-side description of one frame: fp32 or uint16 input; dense results (mask + clean planes) or sparse
// results (bit-plane mask, ascending list of flagged pixels with their replacement values, count).
struct HostFrame {
    const void* img;
    bool u16;
    uint8_t* mask;       // dense results (null: sparse)
    float* clean;
    uint32_t* maskbits;  // sparse results
    int32_t* idx;
    float* val;
    int32_t* count;
    int cap;
};

// one frame through a staging slot: H2D, the path, D2H (slot layout: img | clean | mask | workspace)
// banded: the frame is the only one in flight on this thread's internal copy stream (single-frame entry points), so its
// H2D copy may run there in bands, the first noise/S pass following band by band (hides that pass behind the copy)
int run_host_frame(const HostFrame& io, int h, int w, const lacosmic_params& p, void* slot, cudaStream_t st,
                   bool banded = false) {
    size_t P = (size_t)h * w, plane = align_up(P * 4, 256);
    char* base = (char*)slot;
    float* d_img = (float*)base;
    float* d_clean = (float*)(base + plane);
    uint8_t* d_mask = (uint8_t*)(base + 2 * plane);
    Workspace ws = carve(base + 2 * plane + align_up(P, 256), h, w);
    if (io.u16) {
        // the raw frame is staged in the clean plane, which is dead until the path starts
        uint16_t* d_raw = (uint16_t*)d_clean;
        CK(cudaMemcpyAsync(d_raw, io.img, P * 2, cudaMemcpyHostToDevice, st));
        k_u16_to_f32<<<(unsigned)((P + 2047) / 2048), 256, 0, st>>>(d_raw, d_img, P);
        LAUNCHED();
    }
    BandSync bands;
    BatchStreams* bs = nullptr;
    int nb = 0;
    if (!io.u16 && banded && p.mode == LACOSMIC_MODE_LAZY && p.niter > 0 && p.gain != 0.0f &&
        (nb = band_plan(h, w, bands.row_end, bands.upto)) > 0 && (bs = batch_streams())) {
        const float* src = (const float*)io.img;
        CK(cudaEventRecord(bs->fork, st));                 // the slot is free once the caller's earlier work is done
        CK(cudaStreamWaitEvent(bs->copy, bs->fork, 0));
        int r0 = 0;
        for (int b = 0; b < nb; ++b) {
            const int r1 = bands.row_end[b];
            CK(cudaMemcpyAsync(d_img + (size_t)r0 * w, src + (size_t)r0 * w, (size_t)(r1 - r0) * w * 4, cudaMemcpyHostToDevice, bs->copy));
            CK(cudaEventRecord(bs->band[b], bs->copy));
            bands.ready[b] = bs->band[b];
            r0 = r1;
        }
        bands.n = nb;
    } else if (!io.u16) {
        CK(cudaMemcpyAsync(d_img, io.img, P * 4, cudaMemcpyHostToDevice, st));
    }
    int rc = run_frame(d_img, h, w, p, io.mask ? d_mask : nullptr, d_clean, ws, nullptr, nullptr, st, nullptr,
                       bands.n ? &bands : nullptr);
    if (rc) return rc;
    if (io.mask) {
        CK(cudaMemcpyAsync(io.clean, d_clean, P * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(io.mask, d_mask, P, cudaMemcpyDeviceToHost, st));
        return LACOSMIC_OK;
    }
    // sparse results.  The S plane, the candidate list and the quad list are dead now: values, indices, block sums
    const int cap = (int)std::min<size_t>((size_t)io.cap, P);
    const uint32_t* C = ws.C[p.niter & 1];
    const int wpr = words_per_row(w), nwords = h * wpr;
    const int nblocks = (nwords + lac::CP_WORDS_PER_CTA - 1) / lac::CP_WORDS_PER_CTA;
    int* blocksum = ws.qlist;
    if ((size_t)(nblocks + 1) > (size_t)h * ((w + 3) / 4)) blocksum = (int*)ws.G1;   // tiny frames: any dead plane
    lac::k_popc_blocks<<<nblocks, 256, 0, st>>>(C, nwords, blocksum);
    LAUNCHED();
    lac::k_scan_blocks<<<1, 256, 0, st>>>(blocksum, nblocks);
    LAUNCHED();
    lac::k_emit_flagged<<<nblocks, 256, 0, st>>>(C, nwords, blocksum, d_clean, ws.clist, ws.S, cap, w, wpr);
    LAUNCHED();
    CK(cudaMemcpyAsync(io.maskbits, C, (size_t)nwords * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(io.count, blocksum + nblocks, 4, cudaMemcpyDeviceToHost, st));
    if (cap > 0) {
        CK(cudaMemcpyAsync(io.idx, ws.clist, (size_t)cap * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(io.val, ws.S, (size_t)cap * 4, cudaMemcpyDeviceToHost, st));
    }
    return LACOSMIC_OK;
}

// n host frames through k staging slots on the internal streams (fork / join around the caller's stream)
template <class FrameOf>
int run_host_stream(int n, int h, int w, const lacosmic_params* params, void* dev_workspace, size_t dev_workspace_bytes,
                    cudaStream_t caller, FrameOf frame_of) {
    const size_t slot = align_up(lacosmic_host_workspace_bytes(h, w), 256);
    const int k = (int)std::min<size_t>(std::min(n, LACOSMIC_MAX_BATCH_STREAMS), dev_workspace_bytes / slot);
    if (k < 1) return LACOSMIC_ERR_WORKSPACE;
    BatchStreams* bs = nullptr;
    if (k > 1) {
        bs = batch_streams();
        if (!bs) return LACOSMIC_ERR_CUDA;
        CK(cudaEventRecord(bs->fork, caller));
        for (int s = 0; s < k; ++s) CK(cudaStreamWaitEvent(bs->st[s], bs->fork, 0));
    }
    int rc = LACOSMIC_OK;
    for (int f = 0; f < n; ++f) {
        const int s = f % k;
        rc = run_host_frame(frame_of(f), h, w, params[f], (char*)dev_workspace + (size_t)s * slot,
                            k > 1 ? bs->st[s] : caller);
        if (rc) break;
    }
    if (k > 1) {   // join, also after an error
        for (int s = 0; s < k; ++s) {
            if (!cuda_ok(cudaEventRecord(bs->join[s], bs->st[s])) ||
                !cuda_ok(cudaStreamWaitEvent(caller, bs->join[s], 0)))
                rc = rc ? rc : LACOSMIC_ERR_CUDA;
        }
    }
    return rc;
}
}  // namespace
}  // extern "C++"

int lacosmic_host_band_plan(int h, int w, int32_t* row_end, int32_t* tile_rows) {
    if (!row_end || !tile_rows) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    int re[MAX_BANDS], up[MAX_BANDS];
    const int n = band_plan(h, w, re, up);
    for (int b = 0; b < n; ++b) row_end[b] = re[b], tile_rows[b] = up[b];
    return n;
}

int lacosmic_run_host(const float* img_host, int h, int w, const lacosmic_params* p,
                      uint8_t* mask_out_host, float* clean_out_host, void* dev_workspace,
                      size_t dev_workspace_bytes, void* stream) {
    g_launches = 0;
    if (!img_host || !p || !mask_out_host || !clean_out_host || !dev_workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((rc = check_params(*p))) return rc;
    if ((uintptr_t)dev_workspace & 255) return LACOSMIC_ERR_ALIGN;
    if (dev_workspace_bytes < lacosmic_host_workspace_bytes(h, w)) return LACOSMIC_ERR_WORKSPACE;
    return run_host_frame(HostFrame{img_host, false, mask_out_host, clean_out_host, nullptr, nullptr, nullptr, nullptr, 0},
                          h, w, *p, dev_workspace, (cudaStream_t)stream, true);
}

int lacosmic_run_host_u16(const uint16_t* img_host, int h, int w, const lacosmic_params* p,
                          uint8_t* mask_out_host, float* clean_out_host, void* dev_workspace,
                          size_t dev_workspace_bytes, void* stream) {
    g_launches = 0;
    if (!img_host || !p || !mask_out_host || !clean_out_host || !dev_workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((rc = check_params(*p))) return rc;
    if (((uintptr_t)dev_workspace & 255) || ((uintptr_t)img_host & 1)) return LACOSMIC_ERR_ALIGN;
    if (dev_workspace_bytes < lacosmic_host_workspace_bytes(h, w)) return LACOSMIC_ERR_WORKSPACE;
    return run_host_frame(HostFrame{img_host, true, mask_out_host, clean_out_host, nullptr, nullptr, nullptr, nullptr, 0},
                          h, w, *p, dev_workspace, (cudaStream_t)stream);
}

int lacosmic_run_host_sparse(const float* img_host, int h, int w, const lacosmic_params* p,
                             uint32_t* maskbits_host, int32_t* idx_host, float* val_host, int32_t* count_host,
                             int capacity, void* dev_workspace, size_t dev_workspace_bytes, void* stream) {
    g_launches = 0;
    if (!img_host || !p || !maskbits_host || !idx_host || !val_host || !count_host || !dev_workspace)
        return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((rc = check_params(*p))) return rc;
    if (capacity < 0) return LACOSMIC_ERR_PARAM;
    if ((uintptr_t)dev_workspace & 255) return LACOSMIC_ERR_ALIGN;
    if (dev_workspace_bytes < lacosmic_host_workspace_bytes(h, w)) return LACOSMIC_ERR_WORKSPACE;
    return run_host_frame(HostFrame{img_host, false, nullptr, nullptr, maskbits_host, idx_host, val_host, count_host, capacity},
                          h, w, *p, dev_workspace, (cudaStream_t)stream, true);
}

int lacosmic_run_host_stream_sparse(const void* imgs_host, int input_is_u16, int n, int h, int w,
                                    const lacosmic_params* params, uint32_t* maskbits_host, int32_t* idx_host,
                                    float* val_host, int32_t* counts_host, int capacity, void* dev_workspace,
                                    size_t dev_workspace_bytes, void* stream) {
    g_launches = 0;
    if (n < 0) return LACOSMIC_ERR_SHAPE;
    if (n == 0) return LACOSMIC_OK;
    if (!imgs_host || !params || !maskbits_host || !idx_host || !val_host || !counts_host || !dev_workspace)
        return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    for (int f = 0; f < n; ++f)
        if ((rc = check_params(params[f]))) return rc;
    if (capacity < 0) return LACOSMIC_ERR_PARAM;
    if (((uintptr_t)dev_workspace & 255) || (input_is_u16 && ((uintptr_t)imgs_host & 1))) return LACOSMIC_ERR_ALIGN;
    const size_t P = (size_t)h * w, bw = (size_t)h * words_per_row(w);
    return run_host_stream(n, h, w, params, dev_workspace, dev_workspace_bytes, (cudaStream_t)stream, [&](int f) {
        const void* img = input_is_u16 ? (const void*)((const uint16_t*)imgs_host + f * P)
                                       : (const void*)((const float*)imgs_host + f * P);
        return HostFrame{img, input_is_u16 != 0, nullptr, nullptr, maskbits_host + f * bw,
                         idx_host + (size_t)f * capacity, val_host + (size_t)f * capacity, counts_host + f, capacity};
    });
}

size_t lacosmic_host_batch_workspace_bytes(int h, int w, int concurrency) {
    if (check_shape(h, w) || concurrency < 1) return 0;
    return (size_t)std::min(concurrency, LACOSMIC_MAX_BATCH_STREAMS) * align_up(lacosmic_host_workspace_bytes(h, w), 256);
}

int lacosmic_run_host_batch(const float* imgs_host, int n, int h, int w, const lacosmic_params* params,
                            uint8_t* masks_host, float* cleans_host, void* dev_workspace,
                            size_t dev_workspace_bytes, void* stream) {
    g_launches = 0;
    if (n < 0) return LACOSMIC_ERR_SHAPE;
    if (n == 0) return LACOSMIC_OK;
    if (!imgs_host || !params || !masks_host || !cleans_host || !dev_workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    for (int f = 0; f < n; ++f)
        if ((rc = check_params(params[f]))) return rc;
    if ((uintptr_t)dev_workspace & 255) return LACOSMIC_ERR_ALIGN;
    const size_t P = (size_t)h * w;
    return run_host_stream(n, h, w, params, dev_workspace, dev_workspace_bytes, (cudaStream_t)stream, [&](int f) {
        return HostFrame{imgs_host + f * P, false, masks_host + f * P, cleans_host + f * P, nullptr, nullptr, nullptr,
                         nullptr, 0};
    });
}

// ---- single steps -----------------------------------------------------------------------------

int lacosmic_estimate_gain_ex(const float* img, int h, int w, float readnoise, float* gain_out, float* stats_out,
                              float* path_out, void* workspace, size_t workspace_bytes, void* stream) {
    g_launches = 0;
    if (!img || !gain_out || !workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if (!(readnoise >= 0.0f) || !std::isfinite(readnoise)) return LACOSMIC_ERR_PARAM;
    if (((uintptr_t)img & 15) || ((uintptr_t)workspace & 255)) return LACOSMIC_ERR_ALIGN;
    if (workspace_bytes < lacosmic_workspace_bytes(h, w)) return LACOSMIC_ERR_WORKSPACE;
    Workspace ws = carve(workspace, h, w);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t P = (size_t)h * w;
    // the dense noise/S kernel (generic loader) with the residual plane switched on: r -> clist, med5 -> S
    lac::NoiseArgs ne{ws.S, nullptr, nullptr, nullptr, nullptr, nullptr, h, w, words_per_row(w), 1.0f, 0.0f,
                      1.0f, 1.0f, 0.0f, (float*)ws.clist, nullptr};
    const int ntx = (w + lac::TW - 1) / lac::TW, nt = ntx * ((h + lac::NS_TH - 1) / lac::NS_TH);
    lac::k_noise_S<<<nt, lac::NT, 0, st>>>(img, ne, ntx, nullptr);
    LAUNCHED();
    // the selection kernels write seven floats (six statistics + the path flag) in one block; they go to the tail of the
    // workspace's per-iteration gain array, which a stand-alone estimate does not use, and from there to the caller's
    // two buffers -- so stats_out is six floats, as it has always been documented for this symbol
    float* const seven = (stats_out || path_out) ? ws.gains + 8 : nullptr;
    static_assert(LACOSMIC_MAX_NITER >= 16, "the gain array holds the seven floats at 8..14");
    rc = sigma_clip_gain((const float*)ws.clist, ws.S, P, ws, ws.qlist, (size_t)((char*)ws.C[0] - (char*)ws.qlist) / 4,
                         readnoise * readnoise, gain_out, seven, nullptr, st);
    if (rc) return rc;
    if (stats_out) CK(cudaMemcpyAsync(stats_out, seven, 6 * sizeof(float), cudaMemcpyDeviceToDevice, st));
    if (path_out) CK(cudaMemcpyAsync(path_out, seven + 6, sizeof(float), cudaMemcpyDeviceToDevice, st));
    return LACOSMIC_OK;
}

int lacosmic_estimate_gain(const float* img, int h, int w, float readnoise, float* gain_out, float* stats_out,
                           void* workspace, size_t workspace_bytes, void* stream) {
    return lacosmic_estimate_gain_ex(img, h, w, readnoise, gain_out, stats_out, nullptr, workspace, workspace_bytes, stream);
}

int lacosmic_gain_fast_path_enable(int enable) {
    g_gain_fast.store(enable ? 1 : 0);   // cached graphs are keyed on the switch (GraphKey::gain_fast): none goes stale
    return LACOSMIC_OK;
}

int lacosmic_lplus(const float* in, float* out, int h, int w, void* stream) {
    if (!in || !out) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if (overlap(in, (size_t)h * w * 4, out, (size_t)h * w * 4)) return LACOSMIC_ERR_ALIAS;
    const unsigned nbx = (unsigned)((w + 31) / 32);
    lac::k_lplus<<<nbx * (unsigned)((h + 7) / 8), 256, 0, (cudaStream_t)stream>>>(in, out, h, w, (int)nbx);
    LAUNCHED();
    return LACOSMIC_OK;
}

int lacosmic_medfilt(const float* in, float* out, int h, int w, int k, void* stream) {
    if (!in || !out) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if (k != 3 && k != 5 && k != 7) return LACOSMIC_ERR_PARAM;
    if (overlap(in, (size_t)h * w * 4, out, (size_t)h * w * 4)) return LACOSMIC_ERR_ALIAS;
    const int nbx = (w + lac::TW - 1) / lac::TW;
    const unsigned tg = (unsigned)nbx * (unsigned)((h + lac::TH - 1) / lac::TH);
    dim3 tb(lac::NT);
    cudaStream_t st = (cudaStream_t)stream;
    if (k == 3) lac::k_medfilt<3><<<tg, tb, 0, st>>>(in, out, h, w, nbx);
    else if (k == 5) lac::k_medfilt<5><<<tg, tb, 0, st>>>(in, out, h, w, nbx);
    else lac::k_medfilt<7><<<tg, tb, 0, st>>>(in, out, h, w, nbx);
    LAUNCHED();
    return LACOSMIC_OK;
}

int lacosmic_bitplane_pitch_words(int w) { return w < 1 ? 0 : words_per_row(w); }

int lacosmic_pack_bits(const uint8_t* mask_u8, uint32_t* bits, int h, int w, void* stream) {
    if (!mask_u8 || !bits) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    return pack_bits(mask_u8, bits, h, w, nullptr, (cudaStream_t)stream);
}

int lacosmic_unpack_bits(const uint32_t* bits, uint8_t* mask_u8, int h, int w, void* stream) {
    if (!mask_u8 || !bits) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    return unpack(bits, mask_u8, h, w, (cudaStream_t)stream);
}

int lacosmic_dilate3(const uint32_t* bits_in, uint32_t* bits_out, int h, int w, void* stream) {
    if (!bits_in || !bits_out) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    int wpr = words_per_row(w);
    if (overlap(bits_in, (size_t)h * wpr * 4, bits_out, (size_t)h * wpr * 4)) return LACOSMIC_ERR_ALIAS;
    lac::k_dilate3<<<bit_grid(h, w), 256, 0, (cudaStream_t)stream>>>(bits_in, bits_out, h, w, wpr, bit_nbx(w));
    LAUNCHED();
    return LACOSMIC_OK;
}

int lacosmic_masked_median(const float* img, const uint8_t* mask_u8, float* out, int h, int w,
                           void* workspace, size_t workspace_bytes, void* stream) {
    return lacosmic_masked_median_bpm(img, mask_u8, nullptr, out, h, w, workspace, workspace_bytes, stream);
}

int lacosmic_satstar_mask(const float* img, int h, int w, float satlevel, int grow, uint8_t* out_u8, void* workspace,
                          size_t workspace_bytes, void* stream) {
    g_launches = 0;
    if (!img || !out_u8 || !workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if (std::isnan(satlevel) || grow < 0 || grow > LACOSMIC_MAX_SATGROW) return LACOSMIC_ERR_PARAM;
    if ((uintptr_t)workspace & 255) return LACOSMIC_ERR_ALIGN;
    if (workspace_bytes < lacosmic_workspace_bytes(h, w)) return LACOSMIC_ERR_WORKSPACE;
    Workspace ws = carve(workspace, h, w);
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = satstar_bits(img, h, w, satlevel, grow, ws.NOK, ws.M2, st))) return rc;
    return unpack(ws.NOK, out_u8, h, w, st);
}

int lacosmic_sepmedfilt(const float* in, float* out, float* tmp, int h, int w, int k, void* stream) {
    g_launches = 0;
    if (!in || !out || !tmp) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if (k != 3 && k != 5 && k != 7) return LACOSMIC_ERR_PARAM;
    const size_t B = (size_t)h * w * 4;
    if (overlap(in, B, out, B) || overlap(in, B, tmp, B) || overlap(out, B, tmp, B)) return LACOSMIC_ERR_ALIAS;
    return sepmed(in, out, tmp, h, w, k, (cudaStream_t)stream);
}

size_t lacosmic_sepmed_workspace_bytes(int h, int w) {
    if (check_shape(h, w)) return 0;
    return align_up(lacosmic_workspace_bytes(h, w), 256) + align_up((size_t)h * w * 4, 256);
}

int lacosmic_run_sepmed_compare(const float* img, int h, int w, const lacosmic_params* p, uint8_t* mask_out,
                                float* clean_out, void* workspace, size_t workspace_bytes, int32_t* iter_counts,
                                const lacosmic_debug* dbg, void* stream) {
    g_launches = 0;
    int rc = check_frame_args(img, h, w, p, mask_out, clean_out, workspace, lacosmic_workspace_bytes(h, w));
    if (rc) return rc;
    if (p->gain == 0.0f) return LACOSMIC_ERR_PARAM;      // the comparison path takes a supplied gain only
    if (workspace_bytes < lacosmic_sepmed_workspace_bytes(h, w)) return LACOSMIC_ERR_WORKSPACE;
    if (dbg && (dbg->iter < -1 || dbg->iter >= LACOSMIC_MAX_NITER)) return LACOSMIC_ERR_PARAM;
    if (dbg)   // as in lacosmic_run_ws: fp32 debug planes are written with 16-byte vectors
        for (const float* pl : {dbg->Lp, dbg->N, dbg->S, dbg->Sp, dbg->m3, dbg->F})
            if ((uintptr_t)pl & 15) return LACOSMIC_ERR_ALIGN;
    const size_t P = (size_t)h * w, need = lacosmic_sepmed_workspace_bytes(h, w);
    if (overlap(workspace, need, img, P * 4) || overlap(workspace, need, clean_out, P * 4) || overlap(workspace, need, mask_out, P))
        return LACOSMIC_ERR_ALIAS;
    Workspace ws = carve(workspace, h, w);
    float* third = (float*)((char*)workspace + align_up(ws.bytes, 256));
    return run_sepmed_frame(img, h, w, *p, mask_out, clean_out, ws, third, iter_counts, dbg, (cudaStream_t)stream);
}

int lacosmic_masked_median_bpm(const float* img, const uint8_t* mask_u8, const uint8_t* bpm_u8, float* out, int h, int w,
                               void* workspace, size_t workspace_bytes, void* stream) {
    if (!img || !mask_u8 || !out || !workspace) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((uintptr_t)workspace & 255) return LACOSMIC_ERR_ALIGN;
    if (workspace_bytes < lacosmic_workspace_bytes(h, w)) return LACOSMIC_ERR_WORKSPACE;
    size_t P = (size_t)h * w;
    if (overlap(img, P * 4, out, P * 4)) return LACOSMIC_ERR_ALIAS;
    Workspace ws = carve(workspace, h, w);
    cudaStream_t st = (cudaStream_t)stream;
    const int wpr = words_per_row(w);
    // the fused growth/replacement kernel with M1 = G1 = G2 = mask and C = 0 flags exactly the mask
    // (M2 = dil3(mask) & mask, M3 likewise) and replaces every pixel of it
    if ((rc = lacosmic_pack_bits(mask_u8, ws.M1, h, w, stream))) return rc;
    if (bpm_u8 && (rc = lacosmic_pack_bits(bpm_u8, ws.DONX, h, w, stream))) return rc;
    CK(cudaMemcpyAsync(out, img, P * 4, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemsetAsync(ws.C[0], 0, (size_t)h * wpr * 4, st));
    CK(cudaMemsetAsync(ws.counts, 0, 4, st));
    lac::GrowArgs ga{ws.M1, ws.M1, ws.M1, nullptr, nullptr, nullptr, ws.C[0], ws.C[1], ws.NEED, nullptr, nullptr,
                     nullptr, img, out, ws.counts, 0, h, w, wpr, 0.0f, grow_nbx(w), bpm_u8 ? ws.DONX : nullptr, nullptr, nullptr};
    return grow_replace(ga, nullptr, st);
}

// ---- diagnostics ------------------------------------------------------------------------------

const char* lacosmic_strerror(int code) {
    switch (code) {
        case LACOSMIC_OK: return "ok";
        case LACOSMIC_ERR_NULL: return "required pointer is NULL";
        case LACOSMIC_ERR_SHAPE: return "invalid shape (h, w >= 1 and h*w < 2^31 required)";
        case LACOSMIC_ERR_PARAM: return "invalid parameter";
        case LACOSMIC_ERR_ALIGN: return "pointer not sufficiently aligned";
        case LACOSMIC_ERR_ALIAS: return "buffers overlap";
        case LACOSMIC_ERR_WORKSPACE: return "workspace too small";
        case LACOSMIC_ERR_CUDA: return "CUDA call failed (see lacosmic_last_cuda_error)";
        case LACOSMIC_ERR_TOO_LARGE: return "frame exceeds the built-in scratch (h * ceil(w/32) <= 131072 words); use the workspace variant";
        default: return "unknown error code";
    }
}

int lacosmic_kernel_timing_enable(int enable) {
    if (enable && !g_kt.ev) {
        g_kt.ev = new cudaEvent_t[2 * KTiming::MAXSPANS];
        for (int i = 0; i < 2 * KTiming::MAXSPANS; ++i) CK(cudaEventCreate(&g_kt.ev[i]));
    }
    g_kt.enabled = enable != 0;
    g_kt.n = 0;
    return LACOSMIC_OK;
}

int lacosmic_kernel_timing_read(float* ms_sum, int32_t* spans) {
    if (!ms_sum || !spans) return LACOSMIC_ERR_NULL;
    for (int c = 0; c < KC_COUNT; ++c) ms_sum[c] = 0.0f, spans[c] = 0;
    for (int i = 0; i < g_kt.n; ++i) {
        float ms = 0.0f;
        CK(cudaEventElapsedTime(&ms, g_kt.ev[2 * i], g_kt.ev[2 * i + 1]));
        ms_sum[g_kt.cls[i]] += ms;
        spans[g_kt.cls[i]] += 1;
    }
    g_kt.n = 0;
    return LACOSMIC_OK;
}

const char* lacosmic_kernel_class_name(int cls) {
    static const char* names[KC_COUNT] = {"noise_S", "fine_gates", "grow_replace", "lists", "bits",
                                          "eval_candidates", "noise_S_quads", "gain_select", "whole_frame"};
    return (cls >= 0 && cls < KC_COUNT) ? names[cls] : "?";
}

int lacosmic_probe_minmax_rate(int kind, double* instr_per_s_host, void* stream) {
    if (!instr_per_s_host) return LACOSMIC_ERR_NULL;
    if (kind != 0 && kind != 1) return LACOSMIC_ERR_PARAM;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* sink = nullptr;
    CK(cudaMalloc(&sink, 256));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = LACOSMIC_OK;
    const int iters = 4096, reps = 3, grid = sms * lac::PROBE_CTAS_PER_SM;
    auto launch = [&]() {
        if (kind == 0) lac::k_probe_minmax<0><<<grid, lac::PROBE_THREADS, 0, st>>>(sink, iters, 1.0009765625f);
        else lac::k_probe_minmax<1><<<grid, lac::PROBE_THREADS, 0, st>>>(sink, iters, 1.0009765625f);
    };
    double best_ms = 0.0;
    if (!cuda_ok(cudaEventCreate(&e0)) || !cuda_ok(cudaEventCreate(&e1))) rc = LACOSMIC_ERR_CUDA;
    if (!rc) launch();   // warm-up
    for (int r = 0; r < reps && !rc; ++r) {
        float ms = 0.0f;
        if (!cuda_ok(cudaEventRecord(e0, st))) { rc = LACOSMIC_ERR_CUDA; break; }
        launch();
        if (!cuda_ok(cudaGetLastError()) || !cuda_ok(cudaEventRecord(e1, st)) || !cuda_ok(cudaEventSynchronize(e1)) ||
            !cuda_ok(cudaEventElapsedTime(&ms, e0, e1))) { rc = LACOSMIC_ERR_CUDA; break; }
        if (r == 0 || ms < best_ms) best_ms = ms;
    }
    if (!rc && best_ms > 0.0) {
        const double instr = (double)grid * lac::PROBE_THREADS * (double)iters * lac::PROBE_STAGES_PER_ITER * 8.0;
        *instr_per_s_host = instr / (best_ms * 1e-3);
    } else if (!rc) {
        rc = LACOSMIC_ERR_CUDA;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    return rc;
}

int lacosmic_stats_enable(int enable) {
    g_stats = enable != 0;
    return LACOSMIC_OK;
}

int lacosmic_frame_stats(const void* workspace, int h, int w, int32_t* stats_host, void* stream) {
    if (!workspace || !stats_host) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((uintptr_t)workspace & 255) return LACOSMIC_ERR_ALIGN;
    Workspace ws = carve(const_cast<void*>(workspace), h, w);
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemcpyAsync(stats_host, ws.counts, (size_t)NCOUNTERS * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return LACOSMIC_OK;
}

int lacosmic_gain_zone_info(const void* workspace, int h, int w, int32_t* info_host, void* stream) {
    if (!workspace || !info_host) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    if ((uintptr_t)workspace & 255) return LACOSMIC_ERR_ALIGN;
    Workspace ws = carve(const_cast<void*>(workspace), h, w);
    static_assert(sizeof(lac::SelZone) <= LACOSMIC_GAIN_ZONE_WORDS * 4, "header and library disagree");
    cudaStream_t st = (cudaStream_t)stream;
    std::memset(info_host, 0, LACOSMIC_GAIN_ZONE_WORDS * 4);
    CK(cudaMemcpyAsync(info_host, ws.zone, sizeof(lac::SelZone), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return LACOSMIC_OK;
}

int lacosmic_last_cuda_error(void) { return g_last_cuda_error; }
int lacosmic_last_launch_count(void) { return g_launches; }
const char* lacosmic_version(void) { return "lacosmic-b200 0.4 (sm_100a)"; }

}  // extern "C"

// ---- step (7) without any allocation (include/lacosmic.h, lacosmic_masked_median_noalloc) -----------------
// For callers that cannot bring a workspace: the five bit-planes and the counter that lacosmic_masked_median_bpm
// carves out of the caller's workspace live in a fixed array of this library's device image instead.  The array
// exists once per GPU that loads the library and is shared by every call on that GPU.
//
// In host code the NAME of a __device__ array is only a handle for the runtime's symbol functions, not a device
// address; handing `g_noalloc_scratch` itself to a kernel or to cudaMemsetAsync would make the GPU touch unrelated
// memory.  noalloc_scratch() asks the runtime for the real address on the current device and keeps it.
namespace {

constexpr size_t NA_PLANE_WORDS = LACOSMIC_NOALLOC_MAX_WORDS;     // stride between planes: 512 KiB, keeps 256-byte alignment
constexpr int NA_PLANES = 5;                                       // M1, DONX, C[0], C[1], NEED
constexpr size_t NA_WORDS = NA_PLANES * NA_PLANE_WORDS + 64;       // + 256 bytes for the counter
static_assert(NA_WORDS * 4 == LACOSMIC_NOALLOC_SCRATCH_BYTES, "header and library disagree");
static __device__ __align__(256) uint32_t g_noalloc_scratch[NA_WORDS];

// Device address of g_noalloc_scratch on the CURRENT device (nullptr if the look-up fails; the CUDA error is kept for
// lacosmic_last_cuda_error).  One look-up per device, under a lock, with that device current.
uint32_t* noalloc_scratch() {
    static uint32_t* addr[MAX_DEVICES];
    static std::mutex mu;
    int dev = 0;
    if (!cuda_ok(cudaGetDevice(&dev))) return nullptr;
    if (dev < 0 || dev >= MAX_DEVICES) { g_last_cuda_error = (int)cudaErrorInvalidDevice; return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        uint32_t* ptr = nullptr;
        if (!cuda_ok(cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch)) || !ptr) return nullptr;
        addr[dev] = ptr;
    }
    return addr[dev];
}

}  // namespace

extern "C" int lacosmic_masked_median_noalloc(const float* img, const uint8_t* mask_u8, const uint8_t* bpm_u8, float* out,
                                              int h, int w, void* stream) {
    g_launches = 0;
    if (!img || !mask_u8 || !out) return LACOSMIC_ERR_NULL;
    int rc = check_shape(h, w);
    if (rc) return rc;
    const int wpr = words_per_row(w);
    const size_t words = (size_t)h * wpr, P = (size_t)h * w;
    if (words > NA_PLANE_WORDS) return LACOSMIC_ERR_TOO_LARGE;       // nothing enqueued, `out` untouched
    if (overlap(img, P * 4, out, P * 4)) return LACOSMIC_ERR_ALIAS;
    uint32_t* base = noalloc_scratch();                               // first call on this device: the address look-up
    if (!base) return LACOSMIC_ERR_CUDA;
    uint32_t* M1 = base;
    uint32_t* DONX = base + NA_PLANE_WORDS;
    uint32_t* C0 = base + 2 * NA_PLANE_WORDS;
    uint32_t* C1 = base + 3 * NA_PLANE_WORDS;
    uint32_t* NEED = base + 4 * NA_PLANE_WORDS;
    int* count = (int*)(base + NA_PLANES * NA_PLANE_WORDS);
    cudaStream_t st = (cudaStream_t)stream;
    // The array still holds whatever the previous call (any shape, any stream) left in it.  M1 and DONX are written in
    // full by the packing kernels, C1 and NEED by k_grow_replace before anything reads them; what the kernel expects to
    // find at zero -- the old cumulative mask C0 and the counter it adds to -- is cleared here, on every call.
    if ((rc = pack_bits(mask_u8, M1, h, w, nullptr, st))) return rc;
    if (bpm_u8 && (rc = pack_bits(bpm_u8, DONX, h, w, nullptr, st))) return rc;
    CK(cudaMemcpyAsync(out, img, P * 4, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemsetAsync(C0, 0, words * 4, st));
    CK(cudaMemsetAsync(count, 0, 4, st));
    // as in lacosmic_masked_median_bpm: with M1 = G1 = G2 = mask and C = 0 the fused kernel flags exactly the mask and
    // replaces every pixel of it
    lac::GrowArgs ga{M1, M1, M1, nullptr, nullptr, nullptr, C0, C1, NEED, nullptr, nullptr,
                     nullptr, img, out, count, 0, h, w, wpr, 0.0f, grow_nbx(w), bpm_u8 ? DONX : nullptr, nullptr, nullptr};
    return grow_replace(ga, nullptr, st);
}
