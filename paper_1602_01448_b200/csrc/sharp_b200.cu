// sharp_b200.cu -- host side of the C ABI declared in include/sharp_b200.h: the plan (integer geometry, tile
// lists, workspace layout), the iteration schedule and the kernel launches.  All arithmetic of the method runs in
// the kernels of frame_kernel.cuh / object_kernels.cuh; nothing here falls back to the CPU.
#include "../../include/sharp_b200.h"

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "frame_r.cuh"
#include "frame_s.cuh"
#include "object_kernels.cuh"
#include "probe_kernels.cuh"

using namespace sharp;

namespace {

constexpr double kTau = 1e-4;  // reading G4: thr = tau * a_rms
constexpr int kQuadBlocks = 1184;       // grid of the eps_0 reduction (8 blocks per SM on 148 SMs; any device works)
constexpr int kMaxFrameSlots = 1024;   // upper bound on the persistent frame grid (sizes the error partials)
thread_local std::string g_plan_error = "";

size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

}  // namespace

struct sharp_plan_s {
    int m = 0, K = 0, nr = 0, nc = 0;
    bool periodic = false;             // sharp_plan_periodic: frames wrap around the image edges (reading G25)
    int tiles_r = 0, tiles_c = 0;
    std::vector<int32_t> pos;          // K x 2
    std::vector<int32_t> tile_ptr;     // tiles + 1
    std::vector<int32_t> tile_frames;  // CSR entries
    std::string err;

    // device
    bool bound = false;
    cudaStream_t stream = nullptr;
    unsigned char *ws = nullptr;
    size_t ws_bytes = 0;
    int frame_grid = 0;      // persistent CTAs of the frame kernel
    int slots_cap = 0;       // upper bound on frame_grid the workspace was sized for
    int slots_user = 0;      // sharp_set_frame_slots: caps the persistent grid (0 = one CTA per SM slot)
    int sms = 0;             // multiprocessors of the bound device
    int device = -1;         // CUDA device the plan was bound on
    int frame_ctas_max = 0;  // resident CTAs of the iteration kernel on that device
    int frame_nt = 256;
    int sched_sel = 0;       // which of the two schedule counters the next frame launch uses
    int probe_chunk = 64, probe_nchunks = 0;
    int amp_blocks = 0;

    // workspace offsets
    size_t o_a = 0, o_c[2] = {0, 0}, o_psi_z = 0, o_psi_v[2] = {0, 0}, o_den = 0, o_cross = 0, o_w[4] = {0, 0, 0, 0}, o_scratch = 0,
           o_pos = 0, o_tile_ptr = 0, o_tile_frames = 0, o_partials = 0, o_err_partials = 0, o_err_sums = 0, o_pnum = 0,
           o_pden = 0, o_scalars = 0, o_wtmp[3] = {0, 0, 0}, o_wcon = 0, o_pscal = 0, o_quads = 0, o_quad_sum = 0, o_num = 0, o_praw = 0, o_sched = 0, o_total = 0;

    // state
    bool have_I = false, have_probe = false, have_frames = false, have_prev = false;
    int cur = 0, vcur = 0;             // c[cur], psi_v[vcur] are the current factored frames
    bool obj_stale = false;            // den, cross and psi_z do not reflect w_cur yet (deferred after an illumination update)
    bool psi_v_zero = true;            // psi_v[vcur] is identically 0 (z = c)
    bool prev_psi_v_zero = true;
    int w_cur = 0, w_form = 0, w_prev = 0;  // indices into the four probe buffers
    int refine_every = 0;
    // sharded reconstruction: this plan holds a subset of the frames; every sum over frames is
    // completed by the caller's all-reduce before it is used
    sharp_allreduce_fn allreduce = nullptr;
    void *ar_user = nullptr;
    long long K_total = 0;
    int probe_constraint = 0;          // 0 none, 1 Fourier mask m_w, 2 Fourier amplitude a_w
    bool probe_recentre = false;       // centre-of-mass shift after every illumination update
    long long it = 0;
    long long launches = 0;

    // optional per-kernel timing (sharp_profile): CUDA events around the launches of each kernel class
    bool profiling = false;
    struct ProfSpan { int cls; cudaEvent_t beg, end; };
    std::vector<ProfSpan> prof;

    template <class T>
    T *dp(size_t off) const { return reinterpret_cast<T *>(ws + off); }
    size_t npx() const { return (size_t)K * m * m; }
    size_t nobj() const { return (size_t)nr * nc; }
};

namespace {

int fail(sharp_plan_t *p, int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (p) p->err = buf; else g_plan_error = buf;
    return code;
}

int cuda_fail(sharp_plan_t *p, cudaError_t e, const char *what)
{
    return fail(p, SHARP_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

#define CK(call)                                                   \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return cuda_fail(p, e__, #call);   \
    } while (0)

#define CK_LAUNCH(name)                                            \
    do {                                                           \
        cudaError_t e__ = cudaGetLastError();                      \
        if (e__ != cudaSuccess) return cuda_fail(p, e__, name);    \
        ++p->launches;                                             \
    } while (0)

constexpr int kProfMaxSpans = 8192;

// Brackets one launch with events on the plan's stream while profiling is on (no-op otherwise).
struct ProfScope {
    sharp_plan_t *p;
    cudaEvent_t end = nullptr;
    ProfScope(sharp_plan_t *plan, int cls) : p(plan)
    {
        if (!p->profiling || (int)p->prof.size() >= kProfMaxSpans) return;
        cudaEvent_t b = nullptr;
        if (cudaEventCreate(&b) != cudaSuccess || cudaEventCreate(&end) != cudaSuccess) { end = nullptr; return; }
        cudaEventRecord(b, p->stream);
        p->prof.push_back({cls, b, end});
    }
    ~ProfScope() { if (end) cudaEventRecord(end, p->stream); }
};

int grid_for(size_t n, int per_block = 256, int cap = 160 * 16)
{
    size_t b = (n + per_block - 1) / per_block;
    return (int)std::min<size_t>(std::max<size_t>(b, 1), (size_t)cap);
}

// ---- frame kernel dispatch -----------------------------------------------------------------------------------
// m = 64, 128: the register-radix kernel of frame_r.cuh (whole frame on one SM).  m = 256, 512: strips of 8192
// values per CTA, clusters of kCluster256 / kCluster512 CTAs per frame, row<->column transposition through one
// scratch frame per cluster that lives in L2 (frame_s.cuh).
#ifndef SHARP_NT256
#define SHARP_NT256 128
#endif
#ifndef SHARP_CS256
#define SHARP_CS256 8
#endif
constexpr int kNT256 = SHARP_NT256;      // threads per CTA (strip of 32 kNT256 values) at m = 256
#ifndef SHARP_CS512
#define SHARP_CS512 8
#endif
constexpr int kCluster256 = SHARP_CS256, kCluster512 = SHARP_CS512;

// m >= 256: clusters in flight, each owning one scratch frame (m^2 c64) that should stay resident in L2
#ifndef SHARP_SCR512
#define SHARP_SCR512 40
#endif
int max_scratch_clusters(int m) { return m == 256 ? 80 : SHARP_SCR512; }

int cluster_size(int m) { return m <= 128 ? 1 : (m == 256 ? kCluster256 : kCluster512); }

template <class KernelT>
cudaLaunchConfig_t cluster_config(int grid, int nt, int smem, int cs, cudaStream_t st, cudaLaunchAttribute *attr)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(nt);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cs;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cfg;
}

template <class KernelT>
cudaError_t launch_cluster(KernelT kern, int grid, int nt, int smem, int cs, cudaStream_t st, const FrameArgs &a)
{
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = cluster_config<KernelT>(grid, nt, smem, cs, st, attr);
    return cudaLaunchKernelEx(&cfg, kern, a);
}

template <int MODE, bool WRAP>
int frame_dispatch_w(sharp_plan_t *p, const FrameArgs &a, int grid)
{
    ProfScope prof(p, MODE == FRAME_ITER ? SHARP_PROF_FRAME : SHARP_PROF_OTHER);
    switch (p->m) {
    case 64: k_frame_r<64, MODE, WRAP><<<grid, RCfg<64>::NT, RCfg<64>::SMEM_BYTES, p->stream>>>(a); break;
    case 128: k_frame_r<128, MODE, WRAP><<<grid, RCfg<128>::NT, RCfg<128>::SMEM_BYTES, p->stream>>>(a); break;
    case 256:
        CK(launch_cluster(k_frame_s<256, kNT256, MODE, kCluster256, WRAP>, grid, kNT256, SCfg<256, kNT256>::SMEM_BYTES, kCluster256, p->stream, a));
        break;
    case 512:
        CK(launch_cluster(k_frame_s<512, 256, MODE, kCluster512, WRAP>, grid, 256, SCfg<512, 256>::SMEM_BYTES, kCluster512, p->stream, a));
        break;
    default: return fail(p, SHARP_EINVAL, "unsupported frame size %d", p->m);
    }
    CK_LAUNCH("k_frame");
    return SHARP_OK;
}

// the periodic plan runs the WRAP instantiation of the modes that index the object (FRAME_FFT does not)
template <int MODE>
int frame_dispatch(sharp_plan_t *p, const FrameArgs &a, int grid)
{
    if constexpr (MODE != FRAME_FFT) {
        if (p->periodic) return frame_dispatch_w<MODE, true>(p, a, grid);
    }
    return frame_dispatch_w<MODE, false>(p, a, grid);
}

// sets the shared-memory attribute and returns how many CTAs of the kernel can be resident on the device
template <class KernelT>
cudaError_t kernel_prepare(KernelT kern, int nt, int smem, int cs, int sms, int *resident_ctas)
{
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    if (cs > 8) {      // clusters of 16 are beyond the portable size
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    if (cs == 1) {
        int bps = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, nt, smem);
        *resident_ctas = bps * sms;
        return e;
    }
    cudaLaunchAttribute attr[1];
    cudaLaunchConfig_t cfg = cluster_config<KernelT>(sms * 8 / cs * cs, nt, smem, cs, nullptr, attr);
    int nclusters = 0;
    e = cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg);
    *resident_ctas = nclusters * cs;
    return e;
}

template <int MODE, bool WRAP>
cudaError_t frame_prepare_m(int m, int sms, int *resident)
{
    switch (m) {
    case 64: return kernel_prepare(k_frame_r<64, MODE, WRAP>, RCfg<64>::NT, RCfg<64>::SMEM_BYTES, 1, sms, resident);
    case 128: return kernel_prepare(k_frame_r<128, MODE, WRAP>, RCfg<128>::NT, RCfg<128>::SMEM_BYTES, 1, sms, resident);
    case 256: return kernel_prepare(k_frame_s<256, kNT256, MODE, kCluster256, WRAP>, kNT256, SCfg<256, kNT256>::SMEM_BYTES, kCluster256, sms, resident);
    default: return kernel_prepare(k_frame_s<512, 256, MODE, kCluster512, WRAP>, 256, SCfg<512, 256>::SMEM_BYTES, kCluster512, sms, resident);
    }
}

FrameArgs base_frame_args(sharp_plan_t *p)
{
    FrameArgs a;
    memset(&a, 0, sizeof a);
    a.a_int = p->dp<float>(p->o_a);
    a.pos = p->dp<int>(p->o_pos);
    a.scratch = p->dp<float2>(p->o_scratch);
    a.sc = p->dp<DevScalars>(p->o_scalars);
    a.K = p->K;
    a.nr = p->nr;
    a.nc = p->nc;
    // every frame launch consumes one schedule counter and zeroes the other for the launch after it
    a.sched = p->dp<int>(p->o_sched) + p->sched_sel;
    a.sched_next = p->dp<int>(p->o_sched) + (p->sched_sel ^ 1);
    p->sched_sel ^= 1;
    return a;
}

OverlapArgs base_overlap_args(sharp_plan_t *p)
{
    OverlapArgs a;
    memset(&a, 0, sizeof a);
    a.m = p->m; a.nr = p->nr; a.nc = p->nc; a.tiles_c = p->tiles_c;
    a.periodic = p->periodic ? 1 : 0;
    a.pos = p->dp<int>(p->o_pos);
    a.tile_ptr = p->dp<int>(p->o_tile_ptr);
    a.tile_frames = p->dp<int>(p->o_tile_frames);
    a.den = p->dp<float>(p->o_den);
    a.cross = p->dp<float2>(p->o_cross);
    return a;
}

// sum over the ranks of a sharded plan, in place, ordered after the work already enqueued on the plan's stream (the
// caller's function enqueues its collective on that stream); no-op for an ordinary plan
int reduce_over_ranks(sharp_plan_t *p, void *dev_ptr, size_t count, bool is_double)
{
    if (!p->allreduce) return SHARP_OK;
    if (p->allreduce(p->ar_user, dev_ptr, count, is_double ? 1 : 0) != 0)
        return fail(p, SHARP_ECUDA, "the all-reduce callback of the sharded plan failed");
    return SHARP_OK;
}

template <int MODE>
int overlap_launch(sharp_plan_t *p, const OverlapArgs &a_in)
{
    OverlapArgs a = a_in;
    const bool two_step = p->allreduce != nullptr && MODE != OV_DEN && MODE != OV_BLIND;
    if (two_step) a.num_out = p->dp<float2>(p->o_num);
    {
        ProfScope prof(p, (MODE == OV_ITER || MODE == OV_BLIND) ? SHARP_PROF_OVERLAP : SHARP_PROF_OTHER);
        const int grid = p->tiles_r * p->tiles_c;
        switch (p->m) {
        case 64: k_overlap<64, MODE><<<grid, 256, 0, p->stream>>>(a); break;
        case 128: k_overlap<128, MODE><<<grid, 256, 0, p->stream>>>(a); break;
        case 256: k_overlap<256, MODE><<<grid, 256, 0, p->stream>>>(a); break;
        default: k_overlap<512, MODE><<<grid, 256, 0, p->stream>>>(a); break;
        }
    }
    CK_LAUNCH("k_overlap");
    if (MODE == OV_DEN) {
        if (int rc = reduce_over_ranks(p, a.den, p->nobj(), false)) return rc;
        if (a.w_b != nullptr)
            if (int rc = reduce_over_ranks(p, a.cross, 2 * p->nobj(), false)) return rc;
    } else if (two_step) {
        if (int rc = reduce_over_ranks(p, a.num_out, 2 * p->nobj(), false)) return rc;
        ProfScope prof(p, SHARP_PROF_OTHER);
        k_object_epilogue<MODE><<<grid_for(p->nobj()), 256, 0, p->stream>>>(a, a.num_out);
        CK_LAUNCH("k_object_epilogue");
    }
    return SHARP_OK;
}

int rebuild_den(sharp_plan_t *p)
{
    OverlapArgs a = base_overlap_args(p);
    a.w_a = p->dp<float2>(p->o_w[p->w_cur]);
    // the frames may have been formed with another probe: keep sum conj(w_cur) w_form for the re-gather
    a.w_b = (p->have_frames && !p->psi_v_zero) ? p->dp<float2>(p->o_w[p->w_form]) : nullptr;
    return overlap_launch<OV_DEN>(p, a);
}

// psi_z <- L_{w_cur} z for the current factored frames z = c[cur] + w_form . T psi_v[vcur]
int regather_psi_z(sharp_plan_t *p)
{
    OverlapArgs a = base_overlap_args(p);
    a.f = p->dp<float2>(p->o_c[p->cur]);
    a.w_a = p->dp<float2>(p->o_w[p->w_cur]);
    a.w_b = p->dp<float2>(p->o_w[p->w_form]);
    a.psi_z = p->dp<float2>(p->o_psi_z);
    a.psi_v_in = p->psi_v_zero ? nullptr : p->dp<float2>(p->o_psi_v[p->vcur]);
    return overlap_launch<OV_REGATHER>(p, a);
}

// After an illumination update inside sharp_iterate the new Q*Q, the cross term and the re-gathered psi_z are deferred:
// the next iteration's overlap produces them in the same pass (OV_BLIND).  Everything else that reads them calls this.
int ensure_object_state(sharp_plan_t *p)
{
    if (!p->obj_stale) return SHARP_OK;
    p->obj_stale = false;
    if (int rc = rebuild_den(p)) return rc;
    return regather_psi_z(p);
}

// persistent grid of the frame kernels: one CTA (m <= 128) or one cluster (m >= 256) per resident slot, never more
// than there are frames; sharp_set_frame_slots lowers it (tests force several rounds per CTA that way)
void update_frame_grid(sharp_plan_t *p)
{
    const int cs = cluster_size(p->m);
    long long units = std::min<long long>(p->K, p->frame_ctas_max / cs);
    if (cs > 1) units = std::min<long long>(units, max_scratch_clusters(p->m));
    units = std::min<long long>(units, kMaxFrameSlots / cs);
    if (p->slots_user > 0) units = std::min<long long>(units, p->slots_user);
    p->frame_grid = (int)std::max<long long>(1, units) * cs;
}

int free_probe_slot(const sharp_plan_t *p)
{
    for (int j = 0; j < 4; ++j)
        if (j != p->w_cur && j != p->w_form && j != p->w_prev) return j;
    return -1;  // cannot happen: four buffers, three roles
}

// Every entry point that touches the device runs under the device the plan was bound on and restores the caller's
// current device on return (a plan bound on cuda:1 may be driven while cuda:0 is current).
struct DeviceScope {
    int prev = -1;
    explicit DeviceScope(const sharp_plan_t *p)
    {
        if (!p || !p->bound) return;
        int cur = -1;
        if (cudaGetDevice(&cur) == cudaSuccess && cur != p->device && cudaSetDevice(p->device) == cudaSuccess) prev = cur;
    }
    ~DeviceScope() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceScope(const DeviceScope &) = delete;
    DeviceScope &operator=(const DeviceScope &) = delete;
};

// caller device pointers are read and written with 128-bit accesses
bool misaligned(const void *ptr) { return reinterpret_cast<uintptr_t>(ptr) % 16 != 0; }
#define CHECK_ALIGNED(ptr)                                                                              \
    do {                                                                                                \
        if ((ptr) != nullptr && misaligned(ptr)) return fail(p, SHARP_EINVAL, #ptr " must be 16-byte aligned"); \
    } while (0)

int check_ready(sharp_plan_t *p, bool need_I, bool need_probe)
{
    if (!p) return SHARP_EINVAL;
    if (!p->bound) return fail(p, SHARP_ESTATE, "sharp_bind has not been called");
    if (need_I && !p->have_I) return fail(p, SHARP_ESTATE, "sharp_set_intensities has not been called");
    if (need_probe && !p->have_probe) return fail(p, SHARP_ESTATE, "sharp_set_probe has not been called");
    return SHARP_OK;
}

// frames installed directly in c[cur] (z = c): reset the factored state around them
int adopt_frames(sharp_plan_t *p)
{
    if (p->obj_stale) {                  // the old frames are gone: only Q*Q of the current illumination is still owed
        p->obj_stale = false;
        p->have_frames = false;
        if (int rc = rebuild_den(p)) return rc;
    }
    p->psi_v_zero = true;
    p->have_prev = false;
    p->w_form = p->w_cur;
    p->w_prev = p->w_cur;
    p->it = 0;
    p->have_frames = true;
    return regather_psi_z(p);
}

// one m x m transform, out of place, natural order, unitary: the fused frame kernel in FRAME_FFT mode with K = 1
int fft_single(sharp_plan_t *p, const float2 *in, float2 *out, int sign)
{
    FrameArgs fa = base_frame_args(p);
    fa.K = 1;
    fa.c_in = in;
    fa.c_out = out;
    fa.conj_io = (sign == 1);
    return frame_dispatch<FRAME_FFT>(p, fa, cluster_size(p->m));
}

// Step 7 after Eq. 10: Fourier mask or amplitude constraint, then the centre-of-mass shift.
// src (m x m, one of the o_wtmp buffers or a caller buffer) -> dst; src is left unchanged.
int constrain_probe(sharp_plan_t *p, const float2 *src, float2 *dst)
{
    const int mm = p->m * p->m;
    const float2 *cur = src;
    if (p->probe_constraint != 0) {
        float2 *W = p->dp<float2>(p->o_wtmp[1]);
        float2 *back = p->probe_recentre ? p->dp<float2>(p->o_wtmp[2]) : dst;
        if (int rc = fft_single(p, cur, W, -1)) return rc;
        k_probe_fourier<<<mm / 256, 256, 0, p->stream>>>(mm, p->probe_constraint, p->dp<float>(p->o_wcon), p->dp<ProbeScalars>(p->o_pscal), W);
        CK_LAUNCH("k_probe_fourier");
        if (int rc = fft_single(p, W, back, +1)) return rc;
        cur = back;
    }
    if (p->probe_recentre) {
        k_probe_moments<<<1, 256, 0, p->stream>>>(p->m, cur, p->dp<ProbeScalars>(p->o_pscal));
        CK_LAUNCH("k_probe_moments");
        k_cyclic_shift<<<mm / 256, 256, 0, p->stream>>>(p->m, cur, p->dp<ProbeScalars>(p->o_pscal)->shift, dst);
        CK_LAUNCH("k_cyclic_shift");
    } else if (cur != dst) {
        CK(cudaMemcpyAsync(dst, cur, (size_t)mm * 8, cudaMemcpyDeviceToDevice, p->stream));
    }
    return SHARP_OK;
}

}  // namespace

namespace {
// Tiles met by the pixels [x, x + m) of one axis, taken modulo n when the plan is periodic: at most two index ranges
// [lo, hi] (the second one is the wrapped tail).  The periodic plan requires n - m >= TILE - 1, which keeps the two
// ranges disjoint (no tile sees both ends of a frame).
struct TileRanges { int n; int lo[2], hi[2]; };
static TileRanges tile_ranges(int x, int m, int n)
{
    TileRanges t;
    t.n = 1;
    t.lo[0] = x / TILE;
    t.hi[0] = (std::min(x + m, n) - 1) / TILE;
    if (x + m > n) {
        t.n = 2;
        t.lo[1] = 0;
        t.hi[1] = (x + m - n - 1) / TILE;
    }
    return t;
}

static int make_plan(sharp_plan_t **out, int m, int K, const int32_t *pos_rc, int obj_rows, int obj_cols, bool periodic)
{
    if (!out) return fail(nullptr, SHARP_EINVAL, "out is NULL");
    *out = nullptr;
    if (!(m == 64 || m == 128 || m == 256 || m == 512)) return fail(nullptr, SHARP_EINVAL, "m must be 64, 128, 256 or 512 (got %d)", m);
    if (K < 1) return fail(nullptr, SHARP_EINVAL, "K must be >= 1 (got %d)", K);
    if (!pos_rc) return fail(nullptr, SHARP_EINVAL, "pos_rc is NULL");
    if (obj_rows < m || obj_cols < m) return fail(nullptr, SHARP_EINVAL, "object %d x %d smaller than the frame %d", obj_rows, obj_cols, m);
    if (periodic && (obj_rows - m < TILE - 1 || obj_cols - m < TILE - 1))
        return fail(nullptr, SHARP_EINVAL, "periodic plan: the object must exceed the frame by at least %d pixels per axis", TILE - 1);
    if ((long long)K * m * m > (1LL << 40) || (long long)obj_rows * obj_cols > (1LL << 31) - 1)
        return fail(nullptr, SHARP_EINVAL, "problem too large");
    for (int i = 0; i < K; ++i) {
        const int r = pos_rc[2 * i], c = pos_rc[2 * i + 1];
        const int rmax = periodic ? obj_rows - 1 : obj_rows - m, cmax = periodic ? obj_cols - 1 : obj_cols - m;
        if (r < 0 || c < 0 || r > rmax || c > cmax)
            return fail(nullptr, SHARP_EINVAL, "position %d = (%d, %d) outside [0, %d] x [0, %d] (PAPER.md:53%s)", i, r, c, rmax, cmax,
                        periodic ? "; periodic boundary, PAPER.md:248" : "");
    }
    sharp_plan_t *p = new (std::nothrow) sharp_plan_s;
    if (!p) return fail(nullptr, SHARP_ENOMEM, "host allocation failed");
    p->m = m; p->K = K; p->nr = obj_rows; p->nc = obj_cols;
    p->periodic = periodic;
    p->pos.assign(pos_rc, pos_rc + 2 * (size_t)K);
    p->tiles_r = (obj_rows + TILE - 1) / TILE;
    p->tiles_c = (obj_cols + TILE - 1) / TILE;

    // CSR tile lists by a two-pass counting sort over frames in ascending index: frame i touches the tiles of
    // tile_ranges(row) x tile_ranges(col).
    const size_t ntiles = (size_t)p->tiles_r * p->tiles_c;
    p->tile_ptr.assign(ntiles + 1, 0);
    auto for_each_tile = [&](int i, auto &&fn) {
        const TileRanges tr = tile_ranges(pos_rc[2 * i], m, obj_rows), tc = tile_ranges(pos_rc[2 * i + 1], m, obj_cols);
        for (int a = 0; a < tr.n; ++a)
            for (int ty = tr.lo[a]; ty <= tr.hi[a]; ++ty)
                for (int b = 0; b < tc.n; ++b)
                    for (int tx = tc.lo[b]; tx <= tc.hi[b]; ++tx) fn((size_t)ty * p->tiles_c + tx);
    };
    for (int i = 0; i < K; ++i) for_each_tile(i, [&](size_t t) { ++p->tile_ptr[t + 1]; });
    for (size_t j = 0; j < ntiles; ++j) p->tile_ptr[j + 1] += p->tile_ptr[j];
    p->tile_frames.resize((size_t)p->tile_ptr[ntiles]);
    {
        std::vector<int32_t> fill(p->tile_ptr.begin(), p->tile_ptr.end() - 1);
        for (int i = 0; i < K; ++i) for_each_tile(i, [&](size_t t) { p->tile_frames[(size_t)fill[t]++] = i; });
    }

    // workspace layout.  The frame kernel is persistent: at most one scratch slot per resident CTA.
    const int slots_cap = kMaxFrameSlots;
    p->slots_cap = slots_cap;
    p->probe_chunk = 32;
    p->probe_nchunks = (K + p->probe_chunk - 1) / p->probe_chunk;
    p->amp_blocks = grid_for(p->npx());
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    p->o_a = take(p->npx() * 4);
    p->o_c[0] = take(p->npx() * 8);
    p->o_c[1] = take(p->npx() * 8);
    p->o_psi_z = take(p->nobj() * 8);
    p->o_psi_v[0] = take(p->nobj() * 8);
    p->o_psi_v[1] = take(p->nobj() * 8);
    p->o_den = take(p->nobj() * 4);
    p->o_cross = take(p->nobj() * 8);
    for (int j = 0; j < 4; ++j) p->o_w[j] = take((size_t)m * m * 8);
    // m <= 128 keeps the frame in shared memory; above, one L2 scratch slot per cluster of CTAs
    const int cs_plan = cluster_size(m);
    p->o_scratch = take(m <= 128 ? 256 : (size_t)std::min(K, max_scratch_clusters(m)) * m * m * 8);
    p->o_pos = take((size_t)K * 2 * 4);
    p->o_tile_ptr = take((ntiles + 1) * 4);
    p->o_tile_frames = take(std::max<size_t>(p->tile_frames.size(), 1) * 4);
    p->o_partials = take((size_t)p->amp_blocks * 8);
    p->o_err_partials = take((size_t)slots_cap * 3 * 8);
    p->o_err_sums = take(3 * 8);
    p->o_pnum = take((size_t)p->probe_nchunks * m * m * 8);
    p->o_pden = take((size_t)p->probe_nchunks * m * m * 4);
    p->o_scalars = take(sizeof(DevScalars));
    for (int j = 0; j < 3; ++j) p->o_wtmp[j] = take((size_t)m * m * 8);
    p->o_wcon = take((size_t)m * m * 4);
    p->o_pscal = take(sizeof(ProbeScalars));
    p->o_quads = take((size_t)kQuadBlocks * 4 * 8);
    p->o_quad_sum = take(4 * 8);
    p->o_num = take(p->nobj() * 8);            // raw object numerator of a sharded plan (summed over ranks in place)
    p->o_praw = take((size_t)m * m * 3 * 4);   // raw Eq. 10 sums (num.x, num.y, den) of a sharded plan
    p->o_sched = take(2 * sizeof(int));        // frame counters of the dynamic schedule (frame_r.cuh)
    p->o_total = o;
    *out = p;
    return SHARP_OK;
}

}  // namespace

// =================================================================================================================
extern "C" {

int sharp_plan(sharp_plan_t **out, int m, int K, const int32_t *pos_rc, int obj_rows, int obj_cols)
{
    return make_plan(out, m, K, pos_rc, obj_rows, obj_cols, false);
}

int sharp_plan_periodic(sharp_plan_t **out, int m, int K, const int32_t *pos_rc, int obj_rows, int obj_cols)
{
    return make_plan(out, m, K, pos_rc, obj_rows, obj_cols, true);
}

void sharp_destroy(sharp_plan_t *p)
{
    if (!p) return;
    for (auto &s : p->prof) { cudaEventDestroy(s.beg); cudaEventDestroy(s.end); }
    delete p;
}

const char *sharp_last_error(const sharp_plan_t *p) { return p ? p->err.c_str() : g_plan_error.c_str(); }

size_t sharp_workspace_bytes(const sharp_plan_t *p) { return p ? p->o_total : 0; }

int sharp_bind(sharp_plan_t *p, void *dev_workspace, size_t bytes, void *cuda_stream)
{
    if (!p) return SHARP_EINVAL;
    if (!dev_workspace) return fail(p, SHARP_EINVAL, "workspace is NULL");
    if (reinterpret_cast<uintptr_t>(dev_workspace) % 256 != 0) return fail(p, SHARP_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < p->o_total) return fail(p, SHARP_ENOMEM, "workspace too small: %zu < %zu bytes", bytes, p->o_total);
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) return fail(p, SHARP_ECUDA, "no CUDA device: %s (this library has no CPU path)", cudaGetErrorString(e));
    p->ws = static_cast<unsigned char *>(dev_workspace);
    p->ws_bytes = bytes;
    p->stream = static_cast<cudaStream_t>(cuda_stream);
    // the plan lives on the device that owns the workspace, whatever device is current now or later
    cudaPointerAttributes pa;
    CK(cudaPointerGetAttributes(&pa, dev_workspace));
    if (pa.type != cudaMemoryTypeDevice) return fail(p, SHARP_EINVAL, "workspace is not device memory");
    int dev = pa.device, sms = 0, prev_dev = -1;
    CK(cudaGetDevice(&prev_dev));
    struct Restore { int d; ~Restore() { if (d >= 0) cudaSetDevice(d); } } restore{prev_dev != dev ? prev_dev : -1};
    if (prev_dev != dev) CK(cudaSetDevice(dev));
    // size the persistent grid from the occupancy of the iteration kernel
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    int resident = 0, resident2 = 0;
    if (p->periodic) CK((frame_prepare_m<FRAME_ITER, true>(p->m, sms, &resident)));
    else CK((frame_prepare_m<FRAME_ITER, false>(p->m, sms, &resident)));
    CK((frame_prepare_m<FRAME_FFT, false>(p->m, sms, &resident2)));
    resident = std::min(resident, resident2);
    if (p->periodic) CK((frame_prepare_m<FRAME_ERR, true>(p->m, sms, &resident2)));
    else CK((frame_prepare_m<FRAME_ERR, false>(p->m, sms, &resident2)));
    resident = std::min(resident, resident2);
    if (resident < 1) return fail(p, SHARP_ECUDA, "frame kernel does not fit on the device");
    p->sms = sms;
    p->device = dev;
    p->frame_ctas_max = resident;
    update_frame_grid(p);
    CK(cudaMemcpyAsync(p->dp<int>(p->o_pos), p->pos.data(), p->pos.size() * 4, cudaMemcpyHostToDevice, p->stream));
    CK(cudaMemcpyAsync(p->dp<int>(p->o_tile_ptr), p->tile_ptr.data(), p->tile_ptr.size() * 4, cudaMemcpyHostToDevice, p->stream));
    if (!p->tile_frames.empty())
        CK(cudaMemcpyAsync(p->dp<int>(p->o_tile_frames), p->tile_frames.data(), p->tile_frames.size() * 4, cudaMemcpyHostToDevice, p->stream));
    CK(cudaMemsetAsync(p->dp<void>(p->o_scalars), 0, sizeof(DevScalars), p->stream));
    CK(cudaMemsetAsync(p->dp<void>(p->o_pscal), 0, sizeof(ProbeScalars), p->stream));
    CK(cudaMemsetAsync(p->dp<void>(p->o_sched), 0, 2 * sizeof(int), p->stream));
    p->sched_sel = 0;
    CK(cudaStreamSynchronize(p->stream));  // the host vectors may be read until here
    p->bound = true;
    p->have_I = p->have_probe = p->have_frames = p->have_prev = false;
    p->obj_stale = false;
    p->cur = p->vcur = 0;
    p->w_cur = p->w_form = p->w_prev = 0;
    p->psi_v_zero = p->prev_psi_v_zero = true;
    p->it = 0;
    return SHARP_OK;
}

int sharp_set_intensities(sharp_plan_t *p, const float *I_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CHECK_ALIGNED(I_dev);
    if (!I_dev) return fail(p, SHARP_EINVAL, "I_dev is NULL");
    k_amplitudes<<<p->amp_blocks, 256, 0, p->stream>>>(p->m, p->K, I_dev, p->dp<float>(p->o_a), p->dp<double>(p->o_partials));
    CK_LAUNCH("k_amplitudes");
    k_scalars<<<1, 32, 0, p->stream>>>(p->amp_blocks, p->dp<double>(p->o_partials), p->K, kTau, p->dp<DevScalars>(p->o_scalars));
    CK_LAUNCH("k_scalars");
    if (p->allreduce) {
        // ||a||^2 and a_rms are those of the whole scan (PAPER.md:196-206 normalise by the global ||a||; reading G4)
        if (int rc = reduce_over_ranks(p, &p->dp<DevScalars>(p->o_scalars)->A2, 1, true)) return rc;
        k_scalars_thr<<<1, 32, 0, p->stream>>>(p->K_total, kTau, p->dp<DevScalars>(p->o_scalars));
        CK_LAUNCH("k_scalars_thr");
    }
    p->have_I = true;
    return SHARP_OK;
}

int sharp_set_probe(sharp_plan_t *p, const float *w_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CHECK_ALIGNED(w_dev);
    if (!w_dev) return fail(p, SHARP_EINVAL, "w_dev is NULL");
    const size_t bytes = (size_t)p->m * p->m * 8;
    if (!p->have_frames) {
        p->obj_stale = false;
        p->w_cur = p->w_form = p->w_prev = 0;
        CK(cudaMemcpyAsync(p->dp<void>(p->o_w[0]), w_dev, bytes, cudaMemcpyDeviceToDevice, p->stream));
        p->have_probe = true;
        return rebuild_den(p);
    }
    // frames exist: they stay as they are (reading G10); only Q, Q* and Q*Q change from now on
    p->obj_stale = false;                // whatever was deferred for the replaced illumination is moot
    const int slot = free_probe_slot(p);  // four buffers, three roles: one is always free
    CK(cudaMemcpyAsync(p->dp<void>(p->o_w[slot]), w_dev, bytes, cudaMemcpyDeviceToDevice, p->stream));
    p->w_cur = slot;
    if (int rc = rebuild_den(p)) return rc;
    return regather_psi_z(p);
}

int sharp_set_object(sharp_plan_t *p, const float *psi_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(psi_dev);
    p->cur = 0; p->vcur = 0;
    k_split<<<grid_for(p->npx() / 2), 256, 0, p->stream>>>(p->m, p->K, p->dp<int>(p->o_pos), p->nr, p->nc,
                                                            reinterpret_cast<const float2 *>(psi_dev),
                                                            p->dp<float2>(p->o_w[p->w_cur]), p->dp<float2>(p->o_c[0]));
    CK_LAUNCH("k_split");
    return adopt_frames(p);
}

int sharp_set_frames(sharp_plan_t *p, const float *z_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(z_dev);
    if (!z_dev) return fail(p, SHARP_EINVAL, "z_dev is NULL");
    p->cur = 0; p->vcur = 0;
    CK(cudaMemcpyAsync(p->dp<void>(p->o_c[0]), z_dev, p->npx() * 8, cudaMemcpyDeviceToDevice, p->stream));
    return adopt_frames(p);
}

int sharp_set_frame_slots(sharp_plan_t *p, int slots)
{
    if (!p) return SHARP_EINVAL;
    if (slots < 0) return fail(p, SHARP_EINVAL, "slots must be >= 0");
    p->slots_user = slots;
    if (p->bound) update_frame_grid(p);
    return SHARP_OK;
}

int sharp_set_probe_refine(sharp_plan_t *p, int every)
{
    if (!p) return SHARP_EINVAL;
    if (every < 0) return fail(p, SHARP_EINVAL, "refine period must be >= 0");
    p->refine_every = every;
    return SHARP_OK;
}

int sharp_iterate(sharp_plan_t *p, int n, float beta)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, true, true)) return rc;
    if (n < 0) return fail(p, SHARP_EINVAL, "n must be >= 0");
    if (!(beta > 0.5f && beta <= 1.0f)) return fail(p, SHARP_EINVAL, "beta must be in (0.5, 1] (PAPER.md:178), got %g", (double)beta);
    if (!p->have_frames)
        if (int rc = sharp_set_object(p, nullptr)) return rc;
    const float mm = (float)p->m * (float)p->m;
    for (int l = 0; l < n; ++l) {
        // (a1-a4, frame half of a6)  c' = beta z + (1 - 2 beta) P_a z,  z = c + w_form . T psi_v
        FrameArgs fa = base_frame_args(p);
        fa.c_in = p->dp<float2>(p->o_c[p->cur]);
        fa.c_out = p->dp<float2>(p->o_c[p->cur ^ 1]);
        fa.psi_v = p->psi_v_zero ? nullptr : p->dp<float2>(p->o_psi_v[p->vcur]);
        fa.w_form = p->dp<float2>(p->o_w[p->w_form]);
        fa.bm = beta / mm;
        fa.om = 1.0f - 2.0f * beta;
        if (int rc = frame_dispatch<FRAME_ITER>(p, fa, p->frame_grid)) return rc;
        // (a5, object half of a6)  psi_y, psi_v' = beta (2 psi_y - psi_z), psi_z' = psi_y
        OverlapArgs oa = base_overlap_args(p);
        oa.f = fa.c_out;
        oa.w_a = p->dp<float2>(p->o_w[p->w_cur]);
        oa.psi_z = p->dp<float2>(p->o_psi_z);
        oa.psi_v_out = p->dp<float2>(p->o_psi_v[p->vcur ^ 1]);
        oa.beta = beta;
        if (p->obj_stale) {
            // the illumination changed after the last iteration: Q*Q, the cross term and L_{w_cur} z come out of this pass
            oa.f_prev = fa.c_in;
            oa.w_b = p->dp<float2>(p->o_w[p->w_form]);
            oa.psi_v_in = p->psi_v_zero ? nullptr : p->dp<float2>(p->o_psi_v[p->vcur]);
            p->obj_stale = false;
            if (int rc = overlap_launch<OV_BLIND>(p, oa)) return rc;
        } else {
            if (int rc = overlap_launch<OV_ITER>(p, oa)) return rc;
        }
        // the new frames are z' = c[cur^1] + w_cur . T psi_v[vcur^1]; the old ones stay readable for eps_Delta
        p->prev_psi_v_zero = p->psi_v_zero;
        p->psi_v_zero = false;
        p->cur ^= 1;
        p->vcur ^= 1;
        p->w_prev = p->w_form;
        p->w_form = p->w_cur;
        p->have_prev = true;
        ++p->it;
        // (a7) illumination refinement, Eq. 10, with psi = psi_y (in psi_z) and the new frames
        if (p->refine_every > 0 && p->it % p->refine_every == 0) {
            const int mm_i = p->m * p->m;
            dim3 g(mm_i / 256, p->probe_nchunks);
            {
                ProfScope prof(p, SHARP_PROF_PROBE);
                k_probe_partial<<<g, 256, 0, p->stream>>>(p->m, p->K, p->probe_chunk, p->dp<int>(p->o_pos), p->nr, p->nc,
                                                          p->dp<float2>(p->o_c[p->cur]), p->dp<float2>(p->o_psi_v[p->vcur]),
                                                          p->dp<float2>(p->o_w[p->w_form]), p->dp<float2>(p->o_psi_z),
                                                          p->dp<float2>(p->o_pnum), p->dp<float>(p->o_pden));
            }
            CK_LAUNCH("k_probe_partial");
            int slot = free_probe_slot(p);
            if (slot < 0) return fail(p, SHARP_ECUDA, "internal: no free probe slot");
            const bool post = p->probe_constraint != 0 || p->probe_recentre;
            float2 *w_eq10 = post ? p->dp<float2>(p->o_wtmp[0]) : p->dp<float2>(p->o_w[slot]);
            float *raw = p->allreduce ? p->dp<float>(p->o_praw) : nullptr;
            k_probe_final<<<mm_i / 256, 256, 0, p->stream>>>(p->m, p->probe_nchunks, p->dp<float2>(p->o_pnum), p->dp<float>(p->o_pden),
                                                             p->dp<float2>(p->o_w[p->w_cur]), w_eq10, raw);
            CK_LAUNCH("k_probe_final");
            if (raw) {
                if (int rc = reduce_over_ranks(p, raw, (size_t)3 * mm_i, false)) return rc;
                k_probe_divide<<<mm_i / 256, 256, 0, p->stream>>>(raw, p->dp<float2>(p->o_w[p->w_cur]), w_eq10);
                CK_LAUNCH("k_probe_divide");
            }
            if (post)
                if (int rc = constrain_probe(p, w_eq10, p->dp<float2>(p->o_w[slot]))) return rc;
            p->w_cur = slot;
            if (p->allreduce) {           // sharded plan: the sums over ranks are taken now
                if (int rc = rebuild_den(p)) return rc;
                if (int rc = regather_psi_z(p)) return rc;
            } else {
                p->obj_stale = true;      // folded into the next iteration's overlap pass (or taken on demand)
            }
        }
    }
    return SHARP_OK;
}

int sharp_get_object(sharp_plan_t *p, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(out_dev);
    if (!out_dev) return fail(p, SHARP_EINVAL, "out_dev is NULL");
    if (!p->have_frames) return fail(p, SHARP_ESTATE, "no frames yet (call sharp_set_object or sharp_iterate)");
    if (int rc = ensure_object_state(p)) return rc;
    CK(cudaMemcpyAsync(out_dev, p->dp<void>(p->o_psi_z), p->nobj() * 8, cudaMemcpyDeviceToDevice, p->stream));
    return SHARP_OK;
}

int sharp_get_probe(sharp_plan_t *p, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(out_dev);
    if (!out_dev) return fail(p, SHARP_EINVAL, "out_dev is NULL");
    CK(cudaMemcpyAsync(out_dev, p->dp<void>(p->o_w[p->w_cur]), (size_t)p->m * p->m * 8, cudaMemcpyDeviceToDevice, p->stream));
    return SHARP_OK;
}

int sharp_get_frames(sharp_plan_t *p, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(out_dev);
    if (!out_dev) return fail(p, SHARP_EINVAL, "out_dev is NULL");
    if (!p->have_frames) return fail(p, SHARP_ESTATE, "no frames yet");
    k_materialize<<<grid_for(p->npx()), 256, 0, p->stream>>>(p->m, p->K, p->dp<int>(p->o_pos), p->nr, p->nc, p->dp<float2>(p->o_c[p->cur]),
                                                             p->psi_v_zero ? nullptr : p->dp<float2>(p->o_psi_v[p->vcur]),
                                                             p->dp<float2>(p->o_w[p->w_form]), reinterpret_cast<float2 *>(out_dev));
    CK_LAUNCH("k_materialize");
    return SHARP_OK;
}

int sharp_get_amplitudes(sharp_plan_t *p, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, true, false)) return rc;
    CHECK_ALIGNED(out_dev);
    if (!out_dev) return fail(p, SHARP_EINVAL, "out_dev is NULL");
    k_amplitudes_natural<<<grid_for(p->npx()), 256, 0, p->stream>>>(p->m, p->K, p->dp<float>(p->o_a), out_dev);
    CK_LAUNCH("k_amplitudes_natural");
    return SHARP_OK;
}

int sharp_errors(sharp_plan_t *p, float out[3])
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, true, true)) return rc;
    if (!out) return fail(p, SHARP_EINVAL, "out is NULL");
    if (!p->have_frames) return fail(p, SHARP_ESTATE, "no frames yet");
    if (int rc = ensure_object_state(p)) return rc;
    FrameArgs fa = base_frame_args(p);
    fa.c_in = p->dp<float2>(p->o_c[p->cur]);
    fa.psi_v = p->psi_v_zero ? nullptr : p->dp<float2>(p->o_psi_v[p->vcur]);
    fa.w_form = p->dp<float2>(p->o_w[p->w_form]);
    if (p->have_prev) {
        fa.c_prev = p->dp<float2>(p->o_c[p->cur ^ 1]);
        fa.psi_v_prev = p->prev_psi_v_zero ? nullptr : p->dp<float2>(p->o_psi_v[p->vcur ^ 1]);
        fa.w_form_prev = p->dp<float2>(p->o_w[p->w_prev]);
    }
    fa.psi_z = p->dp<float2>(p->o_psi_z);
    fa.w_cur = p->dp<float2>(p->o_w[p->w_cur]);
    fa.err_partials = p->dp<double>(p->o_err_partials);
    if (int rc = frame_dispatch<FRAME_ERR>(p, fa, p->frame_grid)) return rc;
    k_sum_triples<<<1, 32, 0, p->stream>>>(p->frame_grid, p->dp<double>(p->o_err_partials), p->dp<double>(p->o_err_sums));
    CK_LAUNCH("k_sum_triples");
    if (int rc = reduce_over_ranks(p, p->dp<double>(p->o_err_sums), 3, true)) return rc;
    double sums[3];
    DevScalars sc;
    CK(cudaMemcpyAsync(sums, p->dp<void>(p->o_err_sums), sizeof sums, cudaMemcpyDeviceToHost, p->stream));
    CK(cudaMemcpyAsync(&sc, p->dp<void>(p->o_scalars), sizeof sc, cudaMemcpyDeviceToHost, p->stream));
    CK(cudaStreamSynchronize(p->stream));
    for (int j = 0; j < 3; ++j) out[j] = (float)sqrt(sums[j] / sc.A2);
    return SHARP_OK;
}

int sharp_sync(sharp_plan_t *p)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CK(cudaStreamSynchronize(p->stream));
    return SHARP_OK;
}

long long sharp_launch_count(const sharp_plan_t *p) { return p ? p->launches : 0; }


int sharp_profile(sharp_plan_t *p, int on)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CK(cudaStreamSynchronize(p->stream));
    for (auto &s : p->prof) { cudaEventDestroy(s.beg); cudaEventDestroy(s.end); }
    p->prof.clear();
    p->profiling = on != 0;
    return SHARP_OK;
}

int sharp_profile_read(sharp_plan_t *p, double ms[SHARP_PROF_NCLASS], long long launches[SHARP_PROF_NCLASS])
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    if (!ms || !launches) return fail(p, SHARP_EINVAL, "NULL argument");
    CK(cudaStreamSynchronize(p->stream));
    for (int j = 0; j < SHARP_PROF_NCLASS; ++j) { ms[j] = 0.0; launches[j] = 0; }
    for (auto &s : p->prof) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, s.beg, s.end));
        ms[s.cls] += (double)t;
        ++launches[s.cls];
    }
    return SHARP_OK;
}

int sharp_tile_grid(const sharp_plan_t *p, int *tiles_r, int *tiles_c)
{
    if (!p || !tiles_r || !tiles_c) return SHARP_EINVAL;
    *tiles_r = p->tiles_r;
    *tiles_c = p->tiles_c;
    return SHARP_OK;
}

int sharp_tile_lists(const sharp_plan_t *p, const int32_t **tile_ptr, const int32_t **tile_frames)
{
    if (!p || !tile_ptr || !tile_frames) return SHARP_EINVAL;
    *tile_ptr = p->tile_ptr.data();
    *tile_frames = p->tile_frames.data();
    return SHARP_OK;
}

int sharp_cover_counts(const sharp_plan_t *p, int32_t *out_host)
{
    if (!p || !out_host) return SHARP_EINVAL;
    // 2-D difference array: +1/-1 at the corners of every rectangle, then prefix sums along both axes; a frame that
    // wraps around an edge of a periodic plan is up to four rectangles
    const int nr = p->nr, nc = p->nc, m = p->m;
    std::vector<int32_t> d((size_t)(nr + 1) * (nc + 1), 0);
    auto at = [&](int r, int c) -> int32_t & { return d[(size_t)r * (nc + 1) + c]; };
    auto rect = [&](int r0, int r1, int c0, int c1) { at(r0, c0) += 1; at(r0, c1) -= 1; at(r1, c0) -= 1; at(r1, c1) += 1; };
    for (int i = 0; i < p->K; ++i) {
        const int r = p->pos[2 * i], c = p->pos[2 * i + 1];
        const int rs[2][2] = {{r, std::min(r + m, nr)}, {0, r + m - nr}}, cs[2][2] = {{c, std::min(c + m, nc)}, {0, c + m - nc}};
        for (int a = 0; a < (r + m > nr ? 2 : 1); ++a)
            for (int b = 0; b < (c + m > nc ? 2 : 1); ++b) rect(rs[a][0], rs[a][1], cs[b][0], cs[b][1]);
    }
    for (int r = 0; r <= nr; ++r)
        for (int c = 1; c <= nc; ++c) at(r, c) += at(r, c - 1);
    for (int r = 1; r <= nr; ++r)
        for (int c = 0; c <= nc; ++c) at(r, c) += at(r - 1, c);
    for (int r = 0; r < nr; ++r)
        for (int c = 0; c < nc; ++c) out_host[(size_t)r * nc + c] = at(r, c);
    return SHARP_OK;
}

int sharp_frame_index(sharp_plan_t *p, long long *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CHECK_ALIGNED(out_dev);
    if (!out_dev) return fail(p, SHARP_EINVAL, "out_dev is NULL");
    k_frame_index<<<grid_for(p->npx()), 256, 0, p->stream>>>(p->m, p->K, p->dp<int>(p->o_pos), p->nr, p->nc, out_dev);
    CK_LAUNCH("k_frame_index");
    return SHARP_OK;
}

int sharp_op_split(sharp_plan_t *p, const float *psi_dev, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(psi_dev);
    CHECK_ALIGNED(out_dev);
    if (!out_dev) return fail(p, SHARP_EINVAL, "out_dev is NULL");
    k_split<<<grid_for(p->npx() / 2), 256, 0, p->stream>>>(p->m, p->K, p->dp<int>(p->o_pos), p->nr, p->nc, reinterpret_cast<const float2 *>(psi_dev),
                                                            p->dp<float2>(p->o_w[p->w_cur]), reinterpret_cast<float2 *>(out_dev));
    CK_LAUNCH("k_split");
    return SHARP_OK;
}

int sharp_op_overlap(sharp_plan_t *p, const float *f_dev, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(f_dev);
    CHECK_ALIGNED(out_dev);
    if (!f_dev || !out_dev) return fail(p, SHARP_EINVAL, "NULL argument");
    if (int rc = ensure_object_state(p)) return rc;
    OverlapArgs a = base_overlap_args(p);
    a.f = reinterpret_cast<const float2 *>(f_dev);
    a.w_a = p->dp<float2>(p->o_w[p->w_cur]);
    a.out = reinterpret_cast<float2 *>(out_dev);
    return overlap_launch<OV_L>(p, a);
}

int sharp_op_pa(sharp_plan_t *p, const float *f_dev, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, true, false)) return rc;
    CHECK_ALIGNED(f_dev);
    CHECK_ALIGNED(out_dev);
    if (!f_dev || !out_dev) return fail(p, SHARP_EINVAL, "NULL argument");
    FrameArgs fa = base_frame_args(p);
    fa.c_in = reinterpret_cast<const float2 *>(f_dev);
    fa.c_out = reinterpret_cast<float2 *>(out_dev);
    fa.bm = 0.0f;  // beta = 0: c' = P_a z
    fa.om = 1.0f;
    return frame_dispatch<FRAME_ITER>(p, fa, p->frame_grid);
}

int sharp_op_fft2(sharp_plan_t *p, const float *f_dev, float *out_dev, int sign)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CHECK_ALIGNED(f_dev);
    CHECK_ALIGNED(out_dev);
    if (!f_dev || !out_dev) return fail(p, SHARP_EINVAL, "NULL argument");
    if (f_dev == out_dev) return fail(p, SHARP_EINVAL, "sharp_op_fft2 is out of place");
    if (sign != 1 && sign != -1) return fail(p, SHARP_EINVAL, "sign must be -1 (F) or +1 (F*)");
    FrameArgs fa = base_frame_args(p);
    fa.c_in = reinterpret_cast<const float2 *>(f_dev);
    fa.c_out = reinterpret_cast<float2 *>(out_dev);
    fa.conj_io = (sign == 1);
    return frame_dispatch<FRAME_FFT>(p, fa, p->frame_grid);
}

int sharp_op_probe(sharp_plan_t *p, const float *psi_dev, const float *z_dev, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(psi_dev);
    CHECK_ALIGNED(z_dev);
    CHECK_ALIGNED(out_dev);
    if (!psi_dev || !z_dev || !out_dev) return fail(p, SHARP_EINVAL, "NULL argument");
    const int mm_i = p->m * p->m;
    dim3 g(mm_i / 256, p->probe_nchunks);
    k_probe_partial<<<g, 256, 0, p->stream>>>(p->m, p->K, p->probe_chunk, p->dp<int>(p->o_pos), p->nr, p->nc,
                                              reinterpret_cast<const float2 *>(z_dev), nullptr, p->dp<float2>(p->o_w[p->w_cur]),
                                              reinterpret_cast<const float2 *>(psi_dev), p->dp<float2>(p->o_pnum), p->dp<float>(p->o_pden));
    CK_LAUNCH("k_probe_partial");
    k_probe_final<<<mm_i / 256, 256, 0, p->stream>>>(p->m, p->probe_nchunks, p->dp<float2>(p->o_pnum), p->dp<float>(p->o_pden),
                                                     p->dp<float2>(p->o_w[p->w_cur]), reinterpret_cast<float2 *>(out_dev), nullptr);
    CK_LAUNCH("k_probe_final");
    return SHARP_OK;
}

int sharp_reconstruct_host(sharp_plan_t *p, const float *I_host, const float *w_host, int n, float beta,
                           float *psi_out_host, float *w_out_host, float eps_out[3])
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    if (!I_host || !w_host) return fail(p, SHARP_EINVAL, "NULL input");
    if (n < 0 || !(beta > 0.5f && beta <= 1.0f)) return fail(p, SHARP_EINVAL, "bad n or beta");
    // staging: the second frame buffer is free until the first iteration writes it
    float *stage = p->dp<float>(p->o_c[1]);
    CK(cudaMemcpyAsync(stage, I_host, p->npx() * 4, cudaMemcpyHostToDevice, p->stream));
    if (int rc = sharp_set_intensities(p, stage)) return rc;
    p->have_frames = false;
    float *wstage = p->dp<float>(p->o_psi_v[1]);  // object-sized >= m*m
    CK(cudaMemcpyAsync(wstage, w_host, (size_t)p->m * p->m * 8, cudaMemcpyHostToDevice, p->stream));
    if (int rc = sharp_set_probe(p, wstage)) return rc;
    if (int rc = sharp_set_object(p, nullptr)) return rc;
    if (int rc = sharp_iterate(p, n, beta)) return rc;
    if (eps_out)
        if (int rc = sharp_errors(p, eps_out)) return rc;
    if (psi_out_host) CK(cudaMemcpyAsync(psi_out_host, p->dp<void>(p->o_psi_z), p->nobj() * 8, cudaMemcpyDeviceToHost, p->stream));
    if (w_out_host) CK(cudaMemcpyAsync(w_out_host, p->dp<void>(p->o_w[p->w_cur]), (size_t)p->m * p->m * 8, cudaMemcpyDeviceToHost, p->stream));
    CK(cudaStreamSynchronize(p->stream));
    return SHARP_OK;
}

// ---- eps_0 against a known solution, default initialisations ----------------------------------
int sharp_eps0(sharp_plan_t *p, const float *psi0_dev, const float *w0_dev, float *out_host)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    CHECK_ALIGNED(psi0_dev);
    CHECK_ALIGNED(w0_dev);
    if (!psi0_dev || !out_host) return fail(p, SHARP_EINVAL, "NULL argument");
    if (!p->have_frames) return fail(p, SHARP_ESTATE, "no frames yet");
    if (int rc = ensure_object_state(p)) return rc;
    const float2 *cross = nullptr;
    if (w0_dev != nullptr) {
        // B = Q* Q_{w0} psi_0 = psi_0 . sum_i conj(w) w0: the cross term the Q*Q kernel already knows how to build
        OverlapArgs a = base_overlap_args(p);
        a.w_a = p->dp<float2>(p->o_w[p->w_cur]);
        a.w_b = reinterpret_cast<const float2 *>(w0_dev);
        if (int rc = overlap_launch<OV_DEN>(p, a)) return rc;
        cross = p->dp<float2>(p->o_cross);
    }
    k_eps0_partial<<<kQuadBlocks, 256, 0, p->stream>>>(p->nobj(), p->dp<float2>(p->o_psi_z), p->dp<float>(p->o_den),
                                                       reinterpret_cast<const float2 *>(psi0_dev), cross, p->dp<double>(p->o_quads));
    CK_LAUNCH("k_eps0_partial");
    k_sum_quads<<<1, 32, 0, p->stream>>>(kQuadBlocks, p->dp<double>(p->o_quads), p->dp<double>(p->o_quad_sum));
    CK_LAUNCH("k_sum_quads");
    double q[4];
    CK(cudaMemcpyAsync(q, p->dp<void>(p->o_quad_sum), sizeof q, cudaMemcpyDeviceToHost, p->stream));
    CK(cudaStreamSynchronize(p->stream));
    const double d2 = q[0] + q[1] - 2.0 * sqrt(q[2] * q[2] + q[3] * q[3]);
    *out_host = q[1] > 0.0 ? (float)sqrt(std::max(d2, 0.0) / q[1]) : 0.0f;
    return SHARP_OK;
}

int sharp_init_probe(sharp_plan_t *p)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, true, false)) return rc;
    const int mm = p->m * p->m;
    double *part = p->dp<double>(p->o_pnum);                // probe_nchunks * m * m * 8 bytes
    dim3 g(mm / 256, p->probe_nchunks);
    k_mean_frame_partial<<<g, 256, 0, p->stream>>>(p->m, p->K, p->probe_chunk, p->dp<float>(p->o_a), part);
    CK_LAUNCH("k_mean_frame_partial");
    k_mean_frame_sum<<<mm / 256, 256, 0, p->stream>>>(p->m, p->probe_nchunks, part);
    CK_LAUNCH("k_mean_frame_sum");
    if (int rc = reduce_over_ranks(p, part, (size_t)mm, true)) return rc;
    k_mean_frame_sqrt<<<mm / 256, 256, 0, p->stream>>>(p->m, p->allreduce ? p->K_total : (long long)p->K, part, p->dp<float2>(p->o_wtmp[0]));
    CK_LAUNCH("k_mean_frame_sqrt");
    if (int rc = fft_single(p, p->dp<float2>(p->o_wtmp[0]), p->dp<float2>(p->o_wtmp[1]), +1)) return rc;
    k_cyclic_shift<<<mm / 256, 256, 0, p->stream>>>(p->m, p->dp<float2>(p->o_wtmp[1]), nullptr, p->dp<float2>(p->o_wtmp[2]));
    CK_LAUNCH("k_cyclic_shift");
    return sharp_set_probe(p, p->dp<float>(p->o_wtmp[2]));
}

int sharp_op_random_object(sharp_plan_t *p, unsigned long long seed, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CHECK_ALIGNED(out_dev);
    if (!out_dev) return fail(p, SHARP_EINVAL, "out_dev is NULL");
    k_random_object<<<grid_for(p->nobj()), 256, 0, p->stream>>>(p->nobj(), seed, reinterpret_cast<float2 *>(out_dev));
    CK_LAUNCH("k_random_object");
    return SHARP_OK;
}

int sharp_init_object_random(sharp_plan_t *p, unsigned long long seed)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, true)) return rc;
    // psi_v[1] is free here: sharp_set_object resets the factored state (psi_v = 0) before anything reads it
    float *tmp = p->dp<float>(p->o_psi_v[1]);
    if (int rc = sharp_op_random_object(p, seed, tmp)) return rc;
    return sharp_set_object(p, tmp);
}

// ---- sharded reconstruction --------------------------------------------------------------------
int sharp_set_sharded(sharp_plan_t *p, sharp_allreduce_fn fn, void *user, long long K_total)
{
    if (!p) return SHARP_EINVAL;
    if (fn != nullptr && K_total < p->K) return fail(p, SHARP_EINVAL, "K_total %lld is smaller than this rank's %d frames", K_total, p->K);
    if (p->have_I || p->have_probe)
        return fail(p, SHARP_ESTATE, "sharp_set_sharded must be called before sharp_set_intensities / sharp_set_probe");
    p->allreduce = fn;
    p->ar_user = user;
    p->K_total = fn ? K_total : 0;
    return SHARP_OK;
}

// ---- illumination constraints and re-centring --------------------------------------------------
int sharp_set_probe_constraint(sharp_plan_t *p, int kind, const float *con_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CHECK_ALIGNED(con_dev);
    if (kind < 0 || kind > 2) return fail(p, SHARP_EINVAL, "constraint kind must be 0 (none), 1 (mask) or 2 (amplitude)");
    if (kind != 0 && !con_dev) return fail(p, SHARP_EINVAL, "con_dev is NULL");
    const int mm = p->m * p->m;
    if (kind != 0) {
        CK(cudaMemcpyAsync(p->dp<void>(p->o_wcon), con_dev, (size_t)mm * 4, cudaMemcpyDeviceToDevice, p->stream));
        k_constraint_scalars<<<1, 256, 0, p->stream>>>(mm, p->dp<float>(p->o_wcon), kTau, p->dp<ProbeScalars>(p->o_pscal));
        CK_LAUNCH("k_constraint_scalars");
    }
    p->probe_constraint = kind;
    return SHARP_OK;
}

int sharp_set_probe_recentre(sharp_plan_t *p, int on)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    p->probe_recentre = on != 0;
    CK(cudaMemsetAsync(p->dp<ProbeScalars>(p->o_pscal)->shift, 0, 4 * sizeof(int), p->stream));
    return SHARP_OK;
}

int sharp_get_probe_shift(sharp_plan_t *p, int32_t last[2], int32_t total[2])
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    ProbeScalars ps;
    CK(cudaMemcpyAsync(&ps, p->dp<void>(p->o_pscal), sizeof ps, cudaMemcpyDeviceToHost, p->stream));
    CK(cudaStreamSynchronize(p->stream));
    if (last) { last[0] = ps.shift[0]; last[1] = ps.shift[1]; }
    if (total) { total[0] = ps.total[0]; total[1] = ps.total[1]; }
    return SHARP_OK;
}

int sharp_op_probe_constrain(sharp_plan_t *p, const float *w_dev, float *out_dev)
{
    DeviceScope dev_scope(p);
    if (int rc = check_ready(p, false, false)) return rc;
    CHECK_ALIGNED(w_dev);
    CHECK_ALIGNED(out_dev);
    if (!w_dev || !out_dev) return fail(p, SHARP_EINVAL, "NULL argument");
    if (w_dev == out_dev) return fail(p, SHARP_EINVAL, "sharp_op_probe_constrain is out of place");
    return constrain_probe(p, reinterpret_cast<const float2 *>(w_dev), reinterpret_cast<float2 *>(out_dev));
}

}  // extern "C"

// ---- allocation-free entry point ------------------------------------------------------------------------------------
// For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it): the batched
// unitary 2-D DFT of 256 x 256 frames with the strip kernel's row<->column transposition scratch in a file-scope device
// array instead of a caller workspace.  The arrays below are held by every GPU that loads the library until exit:
//   g_noalloc_scratch   kNoAllocClusters (16) scratch frames of 256 x 256 c64 = 8 MiB
//   g_noalloc_pos       positions the kernel reads per frame (unused by FRAME_FFT; stay zero), 32 KiB
//   g_noalloc_scalars   DevScalars the kernel reads (unused by FRAME_FFT; stays zero)
// In HOST code these names are host-side stand-ins, not device addresses: the addresses the kernel gets come from
// cudaGetSymbolAddress, once per device, with that device current (noalloc_setup).  Nothing in the scratch has to start at
// zero: stage 1 of every frame writes each scratch element before stage 2 reads it.  All calls share the arrays, so calls
// that overlap on the GPU (different streams, no ordering between them) race.
constexpr int kNoAllocM = 256;
constexpr int kNoAllocClusters = 16;
static_assert(SHARP_NOALLOC_MAX_FRAMES == 4096, "keep include/sharp_b200.h and the static arrays in step");
static __device__ __align__(256) float2 g_noalloc_scratch[(size_t)kNoAllocClusters * kNoAllocM * kNoAllocM];
static __device__ __align__(256) int g_noalloc_pos[2 * SHARP_NOALLOC_MAX_FRAMES];
static __device__ __align__(256) DevScalars g_noalloc_scalars;

namespace {

constexpr int kNoAllocMaxDevices = 64;
struct NoAllocDevice {
    bool ready = false;
    float2 *scratch = nullptr;
    int *pos = nullptr;
    DevScalars *scalars = nullptr;
};
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];

// once per device, with that device current: device addresses of the static arrays, shared-memory opt-in of the kernel
int noalloc_setup(int dev, NoAllocDevice **out)
{
    sharp_plan_t *p = nullptr;      // CK reports through sharp_last_error(NULL)
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(nullptr, SHARP_EINVAL, "device ordinal %d not supported", dev);
    NoAllocDevice &d = g_noalloc_dev[dev];
    if (!d.ready) {
        CK(cudaGetSymbolAddress((void **)&d.scratch, g_noalloc_scratch));
        CK(cudaGetSymbolAddress((void **)&d.pos, g_noalloc_pos));
        CK(cudaGetSymbolAddress((void **)&d.scalars, g_noalloc_scalars));
        CK(cudaFuncSetAttribute(k_frame_s<256, kNT256, FRAME_FFT, kCluster256, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                SCfg<256, kNT256>::SMEM_BYTES));
        d.ready = true;
    }
    *out = &d;
    return SHARP_OK;
}

}  // namespace

extern "C" int sharp_fft2_noalloc(const float *f_dev, float *out_dev, int m, int K, int sign, void *cuda_stream)
{
    sharp_plan_t *p = nullptr;
    if (!f_dev || !out_dev) return fail(nullptr, SHARP_EINVAL, "NULL argument");
    if (f_dev == out_dev) return fail(nullptr, SHARP_EINVAL, "sharp_fft2_noalloc is out of place");
    if (misaligned(f_dev) || misaligned(out_dev)) return fail(nullptr, SHARP_EINVAL, "device pointers must be 16-byte aligned");
    if (m != kNoAllocM) return fail(nullptr, SHARP_EINVAL, "sharp_fft2_noalloc supports m = %d only (got %d)", kNoAllocM, m);
    if (K < 1 || K > SHARP_NOALLOC_MAX_FRAMES)
        return fail(nullptr, SHARP_EINVAL, "sharp_fft2_noalloc: K = %d outside [1, %d] (the static scratch is sized for that many frames)", K,
                    SHARP_NOALLOC_MAX_FRAMES);
    if (sign != 1 && sign != -1) return fail(nullptr, SHARP_EINVAL, "sign must be -1 (F) or +1 (F*)");
    // run on the device that owns the input, whatever device is current
    cudaPointerAttributes pa;
    CK(cudaPointerGetAttributes(&pa, f_dev));
    if (pa.type != cudaMemoryTypeDevice) return fail(nullptr, SHARP_EINVAL, "f_dev is not device memory");
    int prev = -1;
    CK(cudaGetDevice(&prev));
    struct Restore { int d; ~Restore() { if (d >= 0) cudaSetDevice(d); } } restore{prev != pa.device ? prev : -1};
    if (prev != pa.device) CK(cudaSetDevice(pa.device));
    NoAllocDevice *d = nullptr;
    if (int rc = noalloc_setup(pa.device, &d)) return rc;

    FrameArgs a;
    memset(&a, 0, sizeof a);
    a.c_in = reinterpret_cast<const float2 *>(f_dev);
    a.c_out = reinterpret_cast<float2 *>(out_dev);
    a.scratch = d->scratch;          // the device address, NOT the symbol's host-side name
    a.pos = d->pos;
    a.sc = d->scalars;
    a.K = K;
    a.conj_io = (sign == 1);
    const int clusters = std::min(K, kNoAllocClusters);
    CK(launch_cluster(k_frame_s<256, kNT256, FRAME_FFT, kCluster256, false>, clusters * kCluster256, kNT256, SCfg<256, kNT256>::SMEM_BYTES,
                      kCluster256, static_cast<cudaStream_t>(cuda_stream), a));
    CK(cudaGetLastError());
    return SHARP_OK;
}
