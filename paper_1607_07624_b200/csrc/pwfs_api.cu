// pwfs_api.cu -- C ABI of libpwfs.so (include/pwfs.h): parameter validation,
// host-side table construction (double precision), scratch management, kernel
// dispatch and instrumentation.  No torch types, no cuFFT, no CPU fallback: every
// step of the path runs in the kernels of pwfs_kernels.cuh.
#include "../../include/pwfs.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "device_guard.cuh"
#include "pwfs_launch.cuh"

using namespace pwk;

namespace {

constexpr double kTwoPi = 6.283185307179586476925286766559;

// One kernel family per grid size M = 32 R1 (pwfs_launch.cuh); each is instantiated in its own
// translation unit (pwfs_inst.cu compiled with -DPWFS_INST_R1=<R1>) so that the build runs in parallel.
bool find_launcher(int M, bool quarter, Launcher *out) {
    if (M % 32) return false;
    switch (M / 32) {
#define PWFS_CASE(R) case R: *out = launcher_for<R>(quarter); return true;
        PWFS_FOR_EACH_R1(PWFS_CASE)
#undef PWFS_CASE
        default: return false;
    }
}

struct TimedSpan { cudaEvent_t a, b; int cls; };

}  // namespace

struct pwfs {
    pwfs_params prm;
    int device = 0;
    int s = 0;
    bool quarter = false;                    // s == M/4 and no field stop: table-free mask kernels
    std::vector<double> list_dx, list_dy, list_w;   // f3: weighted tilt list (empty: the circle of prm)
    double stop_h = -1.0;                    // f3: square field stop half-width [focal bins], < 0 none
    Launcher L{};
    DevTables tab{};
    std::vector<void *> dev_allocs;          // table memory
    std::vector<uint8_t> valid;              // host copy of the valid mask
    // scratch
    float2 *T = nullptr; size_t T_elems = 0;
    float *colbin = nullptr; size_t colbin_elems = 0;
    float *nsum = nullptr; size_t nsum_elems = 0;      // [F][D] per-column sums over valid detector pixels
    // fused small-grid kernel (M = 128): partial frames, per-frame completion counters
    float *spart = nullptr; unsigned *scount = nullptr; size_t small_frames = 0;
    int small_mode = -1;                               // PWFS_SMALL: 0 never, 1 whenever possible, -1 by batch size
    // host-buffer path
    cudaStream_t hstream = nullptr, in_stream = nullptr, out_stream = nullptr;   // compute, H2D, D2H
    std::vector<cudaEvent_t> in_ev, done_ev, tail_ev;                            // per chunk
    float *d_phase = nullptr, *d_frames = nullptr, *d_slopes = nullptr;
    size_t d_cap_frames = 0;
    // schedule
    int user_fpc = 0, user_ksplit = 0;
    int num_sms = 148;
    int x_resident_ctas = 296, y_resident_warps = 1184;   // what the device holds at once (occupancy query at create)
    size_t scratch_budget = (size_t)32 << 30;   // of the 180 GB; PWFS_SCRATCH_MB overrides
    // instrumentation
    int timing = 0;
    std::vector<TimedSpan> spans;
    std::vector<cudaEvent_t> event_pool;
    float ms_acc[PWFS_NUM_KERNEL_CLASSES] = {0, 0, 0, 0, 0};
    int64_t launches[PWFS_NUM_KERNEL_CLASSES] = {0, 0, 0, 0, 0};
    int last_cuda = 0;
    int last_kernel = -1;                    // kernel class of the last launch that failed, -1 none
    bool debug_only = false;                 // pwfs_debug_create with relaxed window checks: pwfs_debug_intensity only
};

namespace {

#define PWFS_CUDA(h, call)                                         \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) { (h)->last_cuda = (int)e__; return PWFS_ECUDA; } \
    } while (0)

template <typename T>
int upload(pwfs *h, const std::vector<T> &v, const T **dst) {
    void *d = nullptr;
    size_t bytes = std::max<size_t>(v.size(), 1) * sizeof(T);
    cudaError_t e = cudaMalloc(&d, bytes);
    if (e != cudaSuccess) { h->last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }
    h->dev_allocs.push_back(d);
    if (!v.empty()) {
        e = cudaMemcpy(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { h->last_cuda = (int)e; return PWFS_ECUDA; }
    }
    *dst = (const T *)d;
    return PWFS_OK;
}

// Area-overlap rebin tables for one axis (O7): detector bin jj = q*n_sub + i takes
// source px p in [floor(i N / n_sub), ceil((i+1) N / n_sub)) of window q with weight
// |[p,p+1) n [i b,(i+1) b)| = integer / n_sub; `start` is the grid coordinate of the
// first source px in the corner-placed frame used by the kernels.
void build_rebin(int N, int M, int s, int n_sub, std::vector<int> &start, std::vector<int> &cnt,
                 std::vector<float> &w, int &cmax, double yscale) {
    const int D = 2 * n_sub;
    std::vector<std::vector<double>> ws(D);
    start.assign(D, 0); cnt.assign(D, 0); cmax = 0;
    for (int jj = 0; jj < D; ++jj) {
        const int q = jj / n_sub, i = jj % n_sub;
        const long long lo_bin = (long long)i * N, hi_bin = (long long)(i + 1) * N;
        const int p0 = (int)(lo_bin / n_sub);
        const int p1 = (int)((hi_bin + n_sub - 1) / n_sub);     // exclusive
        const int g = q == 0 ? (M - s) % M : s % M;              // window origin, corner-placed grid
        start[jj] = (g + p0) % M;
        for (int p = p0; p < p1; ++p) {
            const long long lo = std::max<long long>((long long)p * n_sub, lo_bin);
            const long long hi = std::min<long long>((long long)(p + 1) * n_sub, hi_bin);
            ws[jj].push_back((double)(hi - lo) / (double)n_sub * yscale);
        }
        cnt[jj] = (int)ws[jj].size();
        cmax = std::max(cmax, cnt[jj]);
    }
    w.assign((size_t)D * cmax, 0.f);
    for (int jj = 0; jj < D; ++jj)
        for (int c = 0; c < cnt[jj]; ++c) w[(size_t)jj * cmax + c] = (float)ws[jj][c];
}

// Valid-subaperture mask (O8): illumination = area-weighted sum of A^2, valid iff
// >= thresh * b^2 * max A^2.  Integer-scaled weights (x n_sub per axis) make every
// term an integer for binary A, so ties at exactly 50 % are decided exactly.
int build_valid(int N, int n_sub, const float *A, double thresh, std::vector<uint8_t> &valid,
                std::vector<int> &vidx) {
    double amax2 = 0.0;
    for (size_t t = 0; t < (size_t)N * N; ++t) amax2 = std::max(amax2, (double)A[t] * (double)A[t]);
    valid.assign((size_t)n_sub * n_sub, 0);
    vidx.clear();
    if (!(amax2 > 0.0)) return 0;
    auto overlap = [&](int i, int p) -> long long {
        long long lo = std::max<long long>((long long)p * n_sub, (long long)i * N);
        long long hi = std::min<long long>((long long)(p + 1) * n_sub, (long long)(i + 1) * N);
        return hi > lo ? hi - lo : 0;
    };
    const double full = (double)N * (double)N * amax2;
    for (int j = 0; j < n_sub; ++j) {
        const int py0 = (int)(((long long)j * N) / n_sub), py1 = (int)((((long long)j + 1) * N + n_sub - 1) / n_sub);
        for (int i = 0; i < n_sub; ++i) {
            const int px0 = (int)(((long long)i * N) / n_sub), px1 = (int)((((long long)i + 1) * N + n_sub - 1) / n_sub);
            double ill = 0.0;
            for (int py = py0; py < py1; ++py)
                for (int px = px0; px < px1; ++px) {
                    const double a = (double)A[(size_t)py * N + px];
                    ill += (double)(overlap(j, py) * overlap(i, px)) * a * a;
                }
            if (ill >= thresh * full) {
                valid[(size_t)j * n_sub + i] = 1;
                vidx.push_back(j * n_sub + i);
            }
        }
    }
    return (int)vidx.size();
}

int build_tables(pwfs *h) {
    const pwfs_params &p = h->prm;
    const bool listed = !h->list_dx.empty();
    const int N = p.n_pupil, M = p.m_grid, K = listed ? (int)h->list_dx.size() : p.mod_points, n_sub = p.n_subap, s = h->s;
    const int R1 = h->L.R1;
    DevTables &t = h->tab;
    t.N = N; t.M = M; t.NP = (N + 31) / 32 * 32; t.K = K;
    t.D = 2 * n_sub; t.n_sub = n_sub; t.slope_norm = p.slope_norm;
    t.t_frames = 0;
#ifdef PWFS_TUNING
    // Tuning builds only (python -m paper_1607_07624_b200.build --tuning -> libpwfs_tuning.so; never in libpwfs.so):
    // PWFS_DEBUG_T_ALIAS=1 makes every frame of a chunk use the T slabs of frame 0, so the row<->column intermediate
    // stays L2-resident -- what the step would cost if T never reached HBM.  The results are WRONG by construction.
    const char *alias = std::getenv("PWFS_DEBUG_T_ALIAS");
    if (alias && alias[0] == '1') t.t_frames = 1;
#endif

    // O0: modulation points; distinct x-tilts (the row pass depends on k only through dx_k)
    // f3: an explicit list (dx, dy, w) replaces the circle; I = sum_k w_k |E_k|^2 / sum_k w_k.  The weight
    // rides on the y-tilt phasor as sqrt(w_k K / sum w), so the kernels and their 1/K scale are unchanged.
    std::vector<double> dx(K), dy(K), ux, amp_k(K, 1.0);
    std::vector<int> jx(K);
    double wsum = 0.0, tmax = (double)p.mod_radius;
    if (listed) {
        for (int k = 0; k < K; ++k) { wsum += h->list_w[k]; tmax = std::max(tmax, std::fabs(h->list_dx[k])); }
        for (int k = 0; k < K; ++k) amp_k[k] = std::sqrt(h->list_w[k] * (double)K / wsum);
    }
    for (int k = 0; k < K; ++k) {
        if (listed) {
            dx[k] = h->list_dx[k];
            dy[k] = h->list_dy[k];
        } else {
            const double th = (double)p.mod_angle0 + kTwoPi * (double)k / (double)K;
            dx[k] = (double)p.mod_radius * std::cos(th);
            dy[k] = (double)p.mod_radius * std::sin(th);
        }
        int found = -1;
        for (size_t u = 0; u < ux.size(); ++u)
            if (std::fabs(ux[u] - dx[k]) <= 1e-9 * std::max(1.0, tmax)) { found = (int)u; break; }
        if (found < 0) { found = (int)ux.size(); ux.push_back(dx[k]); }
        jx[k] = found;
    }
    t.KX = (int)ux.size();
    const double c = 0.5 * (double)(N - 1);
    t.NXP = 32 * ((R1 + 1) / 2);                                      // >= N because M >= 2N
    std::vector<float2> txc((size_t)t.KX * t.NXP, make_float2(0.f, 0.f));   // zero in the padding x >= N
    for (int j = 0; j < t.KX; ++j)
        for (int x = 0; x < N; ++x) {
            double turns = ux[j] * ((double)x - c) / (double)N;       // O1, x part
            turns -= std::nearbyint(turns);
            txc[(size_t)j * t.NXP + x] = make_float2((float)std::cos(kTwoPi * turns), (float)std::sin(kTwoPi * turns));
        }
    std::vector<float2> tyt((size_t)K * t.NP, make_float2(0.f, 0.f));   // zero in the padding y >= N
    for (int k = 0; k < K; ++k)
        for (int y = 0; y < N; ++y) {
            double turns = dy[k] * ((double)y - c) / (double)N;       // O1, y part
            turns -= std::nearbyint(turns);
            tyt[(size_t)k * t.NP + y] = make_float2((float)(amp_k[k] * std::cos(kTwoPi * turns)),
                                                    (float)(amp_k[k] * std::sin(kTwoPi * turns)));
        }
    // twiddles between the two register stages, and the 1-D mask a(u)/M (O4; 1/M = O5's scale per axis)
    std::vector<float2> tw((size_t)R1 * 32), am((size_t)R1 * 32);
    for (int k1 = 0; k1 < R1; ++k1)
        for (int n2 = 0; n2 < 32; ++n2) {
            const double ang = -kTwoPi * (double)((k1 * n2) % M) / (double)M;
            tw[(size_t)k1 * 32 + n2] = make_float2((float)std::cos(ang), (float)std::sin(ang));
            const int u = k1 + R1 * n2;                               // n2 plays k2 here
            const int us = u < M / 2 ? u : u - M;
            const long long num = ((long long)s * std::abs(us)) % M;
            const double am_ang = kTwoPi * (double)num / (double)M;
            // table path only (s != M/4 or a field stop): f3's square stop |u~| <= h is separable too
            const double pass = (h->stop_h >= 0.0 && (double)std::abs(us) > h->stop_h) ? 0.0 : 1.0;
            am[(size_t)k1 * 32 + n2] = make_float2((float)(pass * std::cos(am_ang) / M), (float)(pass * std::sin(am_ang) / M));
        }
    // columns of the pupil plane that fall inside a window (corner-placed grid: origins M-s and s)
    std::vector<int> xc_of_x(M, -1), colx;
    for (int q = 0; q < 2; ++q) {
        const int g = q == 0 ? (M - s) % M : s % M;
        for (int pp = 0; pp < N; ++pp) xc_of_x[(g + pp) % M] = 0;
    }
    for (int x = 0; x < M; ++x)
        if (xc_of_x[x] == 0) { xc_of_x[x] = (int)colx.size(); colx.push_back(x); }
    t.ncols = (int)colx.size();
    // rebin tables (same for both axes; the y copy carries no extra scale)
    std::vector<int> rb_start, rb_cnt;
    std::vector<float> rb_w;
    build_rebin(N, M, s, n_sub, rb_start, rb_cnt, rb_w, t.cmax, 1.0);
    // valid mask
    std::vector<int> vidx;
    const double thr = p.illum_thresh > 0.f ? (double)p.illum_thresh : 0.5;
    t.n_valid = build_valid(N, n_sub, p.pupil_amp, thr, h->valid, vidx);
    if (t.n_valid == 0) return PWFS_EINVAL;

    std::vector<float> amp(p.pupil_amp, p.pupil_amp + (size_t)N * N);
    int rc;
    if ((rc = upload(h, amp, &t.amp))) return rc;
    if ((rc = upload(h, txc, &t.txc))) return rc;
    if ((rc = upload(h, tyt, &t.tyt))) return rc;
    if ((rc = upload(h, jx, &t.jx))) return rc;
    // modulation points ordered by x-tilt: consecutive points of one slab T[f][j] re-use the column in registers
    std::vector<int> korder(K);
    for (int k = 0; k < K; ++k) korder[k] = k;
    std::stable_sort(korder.begin(), korder.end(), [&](int a, int b) { return jx[a] < jx[b]; });
    if ((rc = upload(h, korder, &t.korder))) return rc;
    std::vector<int2> kj(K);   // (k, x-tilt index of k) in that order: one load per modulation point in the column pass
    for (int i = 0; i < K; ++i) kj[i] = make_int2(korder[i], jx[korder[i]]);
    if ((rc = upload(h, kj, &t.kj))) return rc;
    if ((rc = upload(h, tw, &t.tw))) return rc;
    if ((rc = upload(h, am, &t.am))) return rc;
    if ((rc = upload(h, colx, &t.colx))) return rc;
    if ((rc = upload(h, xc_of_x, &t.xc_of_x))) return rc;
    if ((rc = upload(h, rb_start, &t.rb_start))) return rc;
    if ((rc = upload(h, rb_cnt, &t.rb_cnt))) return rc;
    if ((rc = upload(h, rb_w, &t.rb_w))) return rc;
    if ((rc = upload(h, vidx, &t.vidx))) return rc;
    if ((rc = upload(h, h->valid, &t.vmask))) return rc;
    return PWFS_OK;
}

// The most frames one chunk may hold: what the scratch budget (and grid.z) allows, or the caller's pinned chunk size.
size_t max_chunk_frames(const pwfs *h) {
    const DevTables &t = h->tab;
    const size_t T_frame = (size_t)t.KX * t.M * t.NP * sizeof(float2);   // T[f][j][x][y], x over the whole grid
    size_t maxF = std::min<size_t>(65535 /* grid.z */, std::max<size_t>(1, h->scratch_budget / std::max<size_t>(T_frame, 1)));
    if (h->user_fpc > 0) maxF = std::min<size_t>(maxF, (size_t)h->user_fpc);
    return maxF;
}

// Split of the modulation loop for chunks of F frames (a function of F alone).
int ksplit_for(const pwfs *h, int F) {
    const DevTables &t = h->tab;
    const int col_warps = (t.ncols + h->L.NB - 1) / h->L.NB;           // column-pass warps per frame
    const int slots = h->num_sms * 12;                                  // resident warps we aim to fill
    int ks = h->user_ksplit > 0 ? h->user_ksplit : 1;
    if (h->user_ksplit <= 0 && (long long)F * col_warps < 2LL * slots) {
        // too few warps for the machine (small batches, B = 1 in a closed loop): split the modulation loop, >= 4
        // points per warp, choosing the split that minimises (waves of resident warps) x (points per warp + 1);
        // the + 1 stands for a warp's prologue and its y-rebin
        double best = 1e300;
        for (int c = 1; c <= std::max(1, t.K / 4); ++c) {
            const long long warps = (long long)F * col_warps * c;
            const double waves = (double)((warps + h->y_resident_warps - 1) / h->y_resident_warps);
            const double cost = waves * ((t.K + c - 1) / c + 1.0);
            if (cost < best * (1.0 - 1e-9)) { best = cost; ks = c; }
        }
    }
    return std::max(1, std::min(ks, t.K));
}

// Frames per chunk and split of the modulation loop for a batch of B frames.  Chunks are as large as the scratch
// budget allows: every launch
// ends with a partly filled wave of CTAs, so fewer, larger launches waste less of the machine (cfg 4: 13.9 ms per 100
// frames in chunks of 15, 13.4 ms in one chunk).  `min_chunks` > 1 (host-buffer path) keeps at least that many chunks so
// that copies still overlap the kernels.
void schedule(const pwfs *h, int B, int *fpc, int *ksplit, int min_chunks = 1) {
    const size_t maxF = max_chunk_frames(h);
    int F = (int)std::min<size_t>(maxF, (size_t)std::max(B, 1));
    if (h->user_fpc <= 0 && min_chunks > 1 && B >= 2 * min_chunks) F = std::min(F, (B + min_chunks - 1) / min_chunks);
    F = std::max(1, std::min(F, std::max(B, 1)));
    if (h->user_fpc <= 0 && F < B) {          // equal chunks: ceil(B / n) frames for the smallest n that fits
        const int n = (B + F - 1) / F;
        F = (B + n - 1) / n;
    }
    *fpc = F; *ksplit = ksplit_for(h, F);
}

// `st`: the stream the caller is about to enqueue on.  cudaMalloc/cudaFree are not allowed while it is being
// captured into a CUDA graph: a batch that needs more scratch than the handle holds is refused with PWFS_EINVAL
// (pwfs_reserve, or one eager pwfs_run of that size, before the capture avoids it).
int ensure_scratch_elems(pwfs *h, size_t needT, size_t needC, size_t needN, cudaStream_t st = nullptr, bool check_capture = false) {
    if (check_capture && (needT > h->T_elems || needC > h->colbin_elems || needN > h->nsum_elems)) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone) return PWFS_EINVAL;
    }
    if (needT > h->T_elems) {
        if (h->T) cudaFree(h->T);
        h->T = nullptr; h->T_elems = 0;
        cudaError_t e = cudaMalloc((void **)&h->T, needT * sizeof(float2));
        if (e != cudaSuccess) { h->last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }
        h->T_elems = needT;
    }
    if (needN > h->nsum_elems) {
        if (h->nsum) cudaFree(h->nsum);
        h->nsum = nullptr; h->nsum_elems = 0;
        cudaError_t e = cudaMalloc((void **)&h->nsum, needN * sizeof(float));
        if (e != cudaSuccess) { h->last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }
        h->nsum_elems = needN;
    }
    if (needC > h->colbin_elems) {
        if (h->colbin) cudaFree(h->colbin);
        h->colbin = nullptr; h->colbin_elems = 0;
        cudaError_t e = cudaMalloc((void **)&h->colbin, needC * sizeof(float));
        if (e != cudaSuccess) { h->last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }
        h->colbin_elems = needC;
    }
    return PWFS_OK;
}

// scratch of one chunk of F frames whose modulation loop is split `ksplit` ways: T, colbin, nsum [elements]
void scratch_need(const pwfs *h, int F, int ksplit, size_t *needT, size_t *needC, size_t *needN) {
    const DevTables &t = h->tab;
    *needT = (size_t)F * t.KX * t.M * t.NP;
    *needC = (size_t)F * ksplit * t.ncols * t.D;
    *needN = (size_t)F * t.D;
}

int ensure_scratch(pwfs *h, int F, int ksplit, cudaStream_t st = nullptr, bool check_capture = false) {
    size_t needT, needC, needN;
    scratch_need(h, F, ksplit, &needT, &needC, &needN);
    return ensure_scratch_elems(h, needT, needC, needN, st, check_capture);
}

struct SpanGuard {
    pwfs *h; cudaStream_t st; int cls; cudaEvent_t a = nullptr, b = nullptr;
    SpanGuard(pwfs *h_, cudaStream_t st_, int cls_) : h(h_), st(st_), cls(cls_) {
        h->launches[cls]++;
        if (!h->timing) return;
        auto get = [&]() {
            cudaEvent_t e = nullptr;
            if (!h->event_pool.empty()) { e = h->event_pool.back(); h->event_pool.pop_back(); }
            else cudaEventCreate(&e);
            return e;
        };
        a = get(); b = get();
        cudaEventRecord(a, st);
    }
    ~SpanGuard() {
        if (!a) return;
        cudaEventRecord(b, st);
        h->spans.push_back({a, b, cls});
    }
};

// ---- pwfs_run_noalloc: scratch that lives in the library image instead of on the CUDA heap ---------------------
// The fused M = 128 kernel needs two pieces of working memory besides its inputs and outputs: one completion counter
// per frame and one partial detector frame per (frame, modulation point).  pwfs_run takes both from cudaMalloc.  For
// callers that must not enter the CUDA allocator, the same kernel can work out of this fixed array, which the driver
// places in device memory when the module is loaded on a GPU and keeps there until the process exits (about 4 MB on
// every GPU that uses the library, whether or not pwfs_run_noalloc is ever called).
//   bytes [0, 256)        : kNoAllocFrames completion counters (unsigned)
//   bytes [256, 256 + 4Mi): kNoAllocPartFloats floats of partial frames, [frame][k][D][D]
constexpr int kNoAllocFrames = PWFS_NOALLOC_MAX_FRAMES;
constexpr size_t kNoAllocPartFloats = PWFS_NOALLOC_MAX_PART_FLOATS;
constexpr size_t kNoAllocCounterBytes = 256;
static_assert(kNoAllocFrames * sizeof(unsigned) <= kNoAllocCounterBytes, "counters must fit their slot");
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocCounterBytes + kNoAllocPartFloats * sizeof(float)];

// In host code `g_noalloc_scratch` is only a stand-in the runtime uses to look the array up; it is NOT the array's
// device address and must never be handed to a kernel.  The real address differs from GPU to GPU, so it is asked for
// once per device (with that device current) and remembered here.
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mu;
unsigned char *g_noalloc_addr[kNoAllocMaxDevices] = {};

// Caller has made `device` current.  Returns the device address of the array on that GPU in *out.
cudaError_t noalloc_scratch_address(int device, unsigned char **out) {
    *out = nullptr;
    if (device < 0 || device >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_addr[device]) {
        unsigned char *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_noalloc_addr[device] = p;
    }
    *out = g_noalloc_addr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" {

const char *pwfs_strerror(int code) {
    switch (code) {
        case PWFS_OK: return "ok";
        case PWFS_EINVAL: return "invalid argument";
        case PWFS_ENOMEM: return "out of memory";
        case PWFS_ECUDA: return "CUDA runtime error";
        case PWFS_EUNSUPPORTED: return "grid size not supported by this build";
        case PWFS_ELIMIT: return "batch exceeds the fixed scratch of pwfs_run_noalloc";
        default: return "unknown pwfs status";
    }
}

int pwfs_supported_grid(int32_t m_grid) {
    Launcher l;
    return find_launcher(m_grid, false, &l) ? 1 : 0;
}

int pwfs_create(const pwfs_params *p, pwfs_t **out) { return pwfs_create_ex(p, nullptr, out); }

static int create_impl(const pwfs_params *p, const pwfs_ext *x, int s_debug, pwfs_t **out);

int pwfs_create_ex(const pwfs_params *p, const pwfs_ext *x, pwfs_t **out) { return create_impl(p, x, -1, out); }

int pwfs_debug_create(const pwfs_params *p, const pwfs_ext *x, int32_t mask_shift_px, pwfs_t **out) {
    if (mask_shift_px < 0) { if (out) *out = nullptr; return PWFS_EINVAL; }
    return create_impl(p, x, mask_shift_px, out);
}

// s_debug >= 0: the mask shift is taken as given (0 = identity mask) and the window constraints are not checked;
// the handle then serves pwfs_debug_intensity only.
static int create_impl(const pwfs_params *p, const pwfs_ext *x, int s_debug, pwfs_t **out) {
    if (out) *out = nullptr;
    if (!p || !out || !p->pupil_amp) return PWFS_EINVAL;
    const int N = p->n_pupil, M = p->m_grid;
    if (N < 2 || M < 2 * N || (M & 1)) return PWFS_EINVAL;
    const bool listed = x && x->n_tilts > 0;
    if (x && x->n_tilts < 0) return PWFS_EINVAL;
    if (listed) {
        if (!x->tilt_x || !x->tilt_y) return PWFS_EINVAL;
        double wsum = 0.0;
        for (int k = 0; k < x->n_tilts; ++k) {
            if (!std::isfinite(x->tilt_x[k]) || !std::isfinite(x->tilt_y[k])) return PWFS_EINVAL;
            const float w = x->tilt_w ? x->tilt_w[k] : 1.f;
            if (!(w >= 0.f) || !std::isfinite(w)) return PWFS_EINVAL;
            wsum += (double)w;
        }
        if (!(wsum > 0.0)) return PWFS_EINVAL;
    } else if (p->mod_points < 1 || !(p->mod_radius >= 0.f) || !std::isfinite(p->mod_radius) || !std::isfinite(p->mod_angle0))
        return PWFS_EINVAL;
    if (x && std::isnan(x->field_stop_px)) return PWFS_EINVAL;
    const double stop_h = (x && x->field_stop_px >= 0.f && (double)x->field_stop_px < 0.5 * M) ? (double)x->field_stop_px : -1.0;
    if (p->n_subap < 1 || p->n_subap > N) return PWFS_EINVAL;
    if (p->slope_norm != 0 && p->slope_norm != 1) return PWFS_EINVAL;
    if (p->illum_thresh > 1.f || !std::isfinite(p->illum_thresh)) return PWFS_EINVAL;
    int s = p->mask_shift_px;
    if (s_debug >= 0) {
        s = s_debug;
        if (s > M / 2) return PWFS_EINVAL;
    } else {
        if (s <= 0) { if (M % 4) return PWFS_EINVAL; s = M / 4; }
        if (2 * s < N || s > M / 2 - N / 2) return PWFS_EINVAL;
    }
    for (size_t i = 0; i < (size_t)N * N; ++i)
        if (!(p->pupil_amp[i] >= 0.f) || !std::isfinite(p->pupil_amp[i])) return PWFS_EINVAL;
    Launcher L;
    const bool quarter = (4 * s == M) && stop_h < 0.0;
    if (!find_launcher(M, quarter, &L)) return PWFS_EUNSUPPORTED;

    pwfs *h = new (std::nothrow) pwfs();
    if (!h) return PWFS_ENOMEM;
    h->prm = *p; h->s = s; h->quarter = quarter; h->L = L; h->device = p->device;
    h->debug_only = s_debug >= 0;
    h->stop_h = stop_h;
    if (listed)
        for (int k = 0; k < x->n_tilts; ++k) {
            h->list_dx.push_back((double)x->tilt_x[k]);
            h->list_dy.push_back((double)x->tilt_y[k]);
            h->list_w.push_back(x->tilt_w ? (double)x->tilt_w[k] : 1.0);
        }
    int rc = PWFS_OK;
    DeviceGuard dg(p->device);
    cudaError_t e = dg.err;
    if (e != cudaSuccess) { h->last_cuda = (int)e; rc = PWFS_ECUDA; }
    if (!rc) {
        cudaDeviceProp prop;
        e = cudaGetDeviceProperties(&prop, p->device);
        if (e != cudaSuccess) { h->last_cuda = (int)e; rc = PWFS_ECUDA; }
        else {
            h->num_sms = prop.multiProcessorCount;
            if (prop.major < 10) rc = PWFS_EUNSUPPORTED;   // built for sm_100a only
        }
    }
    if (!rc) {
        e = cudaFuncSetAttribute(L.xfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem_x);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(L.yfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem_y);
        int nx = 0, ny = 0;
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nx, L.xfn, 32 * L.WPB_X, L.smem_x);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ny, L.yfn, 32 * L.WPB_Y, L.smem_y);
        if (e != cudaSuccess) { h->last_cuda = (int)e; rc = PWFS_ECUDA; }
        h->x_resident_ctas = h->num_sms * std::max(1, nx);
        h->y_resident_warps = h->num_sms * std::max(1, ny) * L.WPB_Y;
    }
    if (!rc && L.sfn) {
        e = cudaFuncSetAttribute(L.sfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem_s);
        if (e != cudaSuccess) { h->last_cuda = (int)e; rc = PWFS_ECUDA; }
        const char *sm = std::getenv("PWFS_SMALL");
        if (sm && (sm[0] == '0' || sm[0] == '1')) h->small_mode = sm[0] - '0';
    }
    if (!rc) {
        const char *env = std::getenv("PWFS_SCRATCH_MB");
        if (env && std::atol(env) > 0) h->scratch_budget = (size_t)std::atol(env) << 20;
        rc = build_tables(h);
    }
    h->prm.pupil_amp = nullptr;   // the caller keeps ownership; we hold a device copy only
    if (rc) { pwfs_destroy(h); return rc; }
    *out = h;
    return PWFS_OK;
}

void pwfs_destroy(pwfs_t *h) {
    if (!h) return;
    DeviceGuard dg(h->device);
    for (void *d : h->dev_allocs) cudaFree(d);
    if (h->T) cudaFree(h->T);
    if (h->colbin) cudaFree(h->colbin);
    if (h->nsum) cudaFree(h->nsum);
    if (h->spart) cudaFree(h->spart);
    if (h->scount) cudaFree(h->scount);
    if (h->d_phase) cudaFree(h->d_phase);
    if (h->d_frames) cudaFree(h->d_frames);
    if (h->d_slopes) cudaFree(h->d_slopes);
    if (h->hstream) cudaStreamDestroy(h->hstream);
    if (h->in_stream) cudaStreamDestroy(h->in_stream);
    if (h->out_stream) cudaStreamDestroy(h->out_stream);
    for (auto ev : h->in_ev) cudaEventDestroy(ev);
    for (auto ev : h->done_ev) cudaEventDestroy(ev);
    for (auto ev : h->tail_ev) cudaEventDestroy(ev);
    for (auto &sp : h->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
    for (auto ev : h->event_pool) cudaEventDestroy(ev);
    delete h;
}

int pwfs_info(const pwfs_t *h, int32_t *det_size, int32_t *n_valid) {
    if (!h) return PWFS_EINVAL;
    if (det_size) *det_size = h->tab.D;
    if (n_valid) *n_valid = h->tab.n_valid;
    return PWFS_OK;
}

int pwfs_valid_mask(const pwfs_t *h, uint8_t *host_mask) {
    if (!h || !host_mask) return PWFS_EINVAL;
    std::memcpy(host_mask, h->valid.data(), h->valid.size());
    return PWFS_OK;
}

int pwfs_last_cuda_error(const pwfs_t *h) { return h ? h->last_cuda : 0; }

int pwfs_last_failed_kernel(const pwfs_t *h) { return h ? h->last_kernel : -1; }

int pwfs_set_schedule(pwfs_t *h, int32_t frames_per_chunk, int32_t k_split) {
    if (!h || frames_per_chunk < 0 || k_split < 0 || k_split > h->tab.K) return PWFS_EINVAL;
    h->user_fpc = frames_per_chunk;
    h->user_ksplit = k_split;
    return PWFS_OK;
}

int pwfs_geometry(const pwfs_t *h, int32_t B, int32_t *n_cols, int32_t *k_unique, int32_t *frames_per_chunk,
                  int32_t *k_split) {
    if (!h) return PWFS_EINVAL;
    int F, ks;
    schedule(h, B, &F, &ks);
    if (n_cols) *n_cols = h->tab.ncols;
    if (k_unique) *k_unique = h->tab.KX;
    if (frames_per_chunk) *frames_per_chunk = F;
    if (k_split) *k_split = ks;
    return PWFS_OK;
}

int pwfs_set_timing(pwfs_t *h, int32_t enable) {
    if (!h) return PWFS_EINVAL;
    h->timing = enable ? 1 : 0;
    return PWFS_OK;
}

int pwfs_get_timing(pwfs_t *h, float ms[PWFS_NUM_KERNEL_CLASSES], int64_t launches[PWFS_NUM_KERNEL_CLASSES]) {
    if (!h) return PWFS_EINVAL;
    for (auto &sp : h->spans) {
        PWFS_CUDA(h, cudaEventSynchronize(sp.b));
        float m = 0.f;
        PWFS_CUDA(h, cudaEventElapsedTime(&m, sp.a, sp.b));
        h->ms_acc[sp.cls] += m;
        h->event_pool.push_back(sp.a);
        h->event_pool.push_back(sp.b);
    }
    h->spans.clear();
    for (int i = 0; i < PWFS_NUM_KERNEL_CLASSES; ++i) {
        if (ms) ms[i] = h->ms_acc[i];
        if (launches) launches[i] = h->launches[i];
        h->ms_acc[i] = 0.f;
        h->launches[i] = 0;
    }
    return PWFS_OK;
}

// A launch that the runtime refuses (bad configuration, sticky fault) is reported at once, with its kernel class.
static int check_launch(pwfs_t *h, int cls) {
    const cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) return PWFS_OK;
    h->last_cuda = (int)e;
    h->last_kernel = cls;
    return PWFS_ECUDA;
}

// One chunk of Fc <= F frames is three enqueue steps: K1 (row pass), K2 (column pass), tail (x-rebin + slopes).
static int launch_k1(pwfs_t *h, const float *d_phase, int Fc, cudaStream_t st) {
    const DevTables &t = h->tab;
    const Launcher &L = h->L;
    SpanGuard g(h, st, 0);   // K1: phasor + x-convolution (a1, a3, a4, a5 along x)
    const int row_ctas = (t.NP + L.RPC - 1) / L.RPC;
    int jsplit = 1;
    if ((long long)row_ctas * Fc >= 2LL * h->x_resident_ctas || t.KX < 6) {
        // split the x-tilt loop only as far as needed to fill the machine (>= 8 waves of 2 CTAs/SM),
        // keeping >= 3 tilts per CTA so the one-off phasor stays amortised
        while ((long long)row_ctas * Fc * jsplit < 16LL * h->num_sms && t.KX / (jsplit + 1) >= 3) ++jsplit;
    } else {   // small batch (less than two waves of CTAs): (waves of resident CTAs) x (x-tilts per CTA + 1 for the
        // phasor), down to ONE tilt per CTA -- with SMs to spare the critical path counts, not the repeated phasor
        // (cfg 2, one frame: 28 CTAs of 4 tilts on 148 SMs ran at 13 % SM-active, profiles/r3_ncu_b1.md)
        double best = 1e300;
        for (int c = 1; c <= t.KX; ++c) {
            const long long ctas = (long long)row_ctas * Fc * c;
            const double waves = (double)((ctas + h->x_resident_ctas - 1) / h->x_resident_ctas);
            const double cost = waves * ((t.KX + c - 1) / c + 1.0);
            if (cost < best * (1.0 - 1e-9)) { best = cost; jsplit = c; }
        }
    }
    L.launch_x(dim3(row_ctas, jsplit, Fc), st, t, d_phase, h->T, jsplit);
    return check_launch(h, 0);
}

static int launch_k2(pwfs_t *h, int Fc, int ks, cudaStream_t st) {
    const DevTables &t = h->tab;
    const Launcher &L = h->L;
    SpanGuard g(h, st, 1);   // K2: y-convolution + |E|^2 over k + y-rebin (a3, a4, a5 along y, a6, a7)
    const int per_cta = L.NB * L.WPB_Y;
    L.launch_y(dim3((t.ncols + per_cta - 1) / per_cta, ks, Fc), st, t, h->T, h->colbin, ks);
    return check_launch(h, 1);
}

static int launch_tail(pwfs_t *h, int Fc, float *d_frames, float *d_slopes, int ks, cudaStream_t st) {
    const DevTables &t = h->tab;
    {   // K3a: x-rebin (a7)
        SpanGuard g(h, st, 2);
        const int threads = std::min(256, (t.D + 31) / 32 * 32);
        // 1/K of O6; the quarter-mask kernels leave O5's 1/M per axis (1/M^4 on |E|^2) to this scale
        const double m4 = h->quarter ? std::pow((double)t.M, 4.0) : 1.0;
        xrebin_kernel<<<dim3(t.D, Fc), threads, 0, st>>>(t, h->colbin, d_frames, h->nsum, ks, (float)(1.0 / ((double)t.K * m4)));
        if (int rc = check_launch(h, 2)) return rc;
    }
    if (d_slopes) {   // K3b: slopes (a8)
        SpanGuard g(h, st, 3);
        slopes_kernel<<<dim3((t.n_valid + 255) / 256, Fc), 256, 0, st>>>(t, d_frames, h->nsum, d_slopes);
        if (int rc = check_launch(h, 3)) return rc;
    }
    return PWFS_OK;
}

// per-chunk events of the two-stream schedule below
static int ensure_chunk_events(pwfs_t *h, size_t n_chunks) {
    while (h->in_ev.size() < n_chunks) {
        cudaEvent_t a, b, c;
        PWFS_CUDA(h, cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
        h->in_ev.push_back(a);
        PWFS_CUDA(h, cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
        h->done_ev.push_back(b);
        PWFS_CUDA(h, cudaEventCreateWithFlags(&c, cudaEventDisableTiming));
        h->tail_ev.push_back(c);
    }
    return PWFS_OK;
}

// The fused kernel serves M = 128 sensors whose pupil, window columns and detector fit its shared-memory plan, when the
// caller has not pinned the schedule; by default for batches that leave the two-kernel path launch-bound.
static bool small_applies(const pwfs_t *h, int B) {
    const DevTables &t = h->tab;
    if (!h->L.launch_s || h->small_mode == 0 || h->user_fpc > 0 || h->user_ksplit > 0) return false;
    if (t.N > 64 || t.ncols > 128 || t.D > 64 || t.cmax > 8) return false;   // SmallCfg::MAXN, MAXCOLS, MAXD, MAXCMAX
    if (h->small_mode == 1) return true;
    return (long long)B * t.K <= 16LL * h->num_sms;
}

static int ensure_small(pwfs_t *h, int B, cudaStream_t st, bool check_capture) {
    if ((size_t)B <= h->small_frames) return PWFS_OK;
    if (check_capture) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone) return PWFS_EINVAL;
    }
    const DevTables &t = h->tab;
    if (h->spart) cudaFree(h->spart);
    if (h->scount) cudaFree(h->scount);
    h->spart = nullptr; h->scount = nullptr; h->small_frames = 0;
    cudaError_t e = cudaMalloc((void **)&h->spart, (size_t)B * t.K * t.D * t.D * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->scount, (size_t)B * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemset(h->scount, 0, (size_t)B * sizeof(unsigned));
    if (e != cudaSuccess) { h->last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }
    h->small_frames = (size_t)B;
    return PWFS_OK;
}

static int run_small(pwfs_t *h, const float *d_phase, int B, float *d_frames, float *d_slopes, cudaStream_t st) {
    const DevTables &t = h->tab;
    const size_t NN = (size_t)t.N * t.N, DD = (size_t)t.D * t.D, SS = (size_t)2 * t.n_valid;
    const double m4 = h->quarter ? std::pow((double)t.M, 4.0) : 1.0;
    for (int f0 = 0; f0 < B; f0 += 65535) {                        // grid.y limit
        const int Fc = std::min(65535, B - f0);
        SpanGuard g(h, st, 4);
        h->L.launch_s(dim3(t.K, Fc), st, t, d_phase + (size_t)f0 * NN, h->spart + (size_t)f0 * t.K * DD,
                      h->scount + f0, d_frames + (size_t)f0 * DD, d_slopes ? d_slopes + (size_t)f0 * SS : nullptr,
                      (float)(1.0 / ((double)t.K * m4)));
        if (int rc = check_launch(h, 4)) return rc;
    }
    return PWFS_OK;
}

// Sizes everything a pwfs_run of ANY batch of 1..B frames can need, not just the schedule of exactly B frames: a
// smaller batch may take the other path (the fused kernel serves small batches only) or split its modulation loop
// further (more colbin per frame), and must find its scratch in place when it is captured into a graph.
int pwfs_reserve(pwfs_t *h, int32_t B) {
    if (!h || B < 1) return PWFS_EINVAL;
    DeviceGuard dg(h->device);
    PWFS_CUDA(h, dg.err);
    if (small_applies(h, 1)) {                    // the fused kernel takes batches of 1..bs frames
        const long long cap = h->small_mode == 1 ? (long long)B : 16LL * h->num_sms / std::max(1, h->tab.K);
        const int bs = (int)std::min<long long>(B, cap);
        if (bs >= 1)
            if (int rc = ensure_small(h, bs, nullptr, false)) return rc;
        if (bs == B) return PWFS_OK;              // ... which is all of them
    }
    // two-kernel path: a batch of b <= B frames runs in chunks of F <= min(b, max_chunk_frames) frames, every such F
    // is some batch's chunk size, and the k-split is a function of F
    const int Fmax = (int)std::min<size_t>((size_t)B, max_chunk_frames(h));
    size_t needT = 0, needC = 0, needN = 0;
    for (int F = 1; F <= Fmax; ++F) {
        size_t nT, nC, nN;
        scratch_need(h, F, ksplit_for(h, F), &nT, &nC, &nN);
        needT = std::max(needT, nT); needC = std::max(needC, nC); needN = std::max(needN, nN);
    }
    int rc = ensure_scratch_elems(h, needT, needC, needN);
    if (rc) return rc;
    int F, ks;
    schedule(h, B, &F, &ks);                      // the largest batch has the most chunks
    const size_t n_chunks = ((size_t)B + F - 1) / F;
    if (n_chunks > 1) {
        if (!h->out_stream) PWFS_CUDA(h, cudaStreamCreateWithFlags(&h->out_stream, cudaStreamNonBlocking));
        if ((rc = ensure_chunk_events(h, n_chunks))) return rc;
    }
    return PWFS_OK;
}

int pwfs_run(pwfs_t *h, const float *d_phase, int32_t B, float *d_frames, float *d_slopes, void *cuda_stream) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_phase || !d_frames || h->debug_only) return PWFS_EINVAL;
    DeviceGuard dg(h->device);
    PWFS_CUDA(h, dg.err);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const DevTables &t = h->tab;
    if (small_applies(h, B)) {                                     // M = 128, small batch: the whole path in one kernel
        if (int rc = ensure_small(h, B, st, true)) return rc;
        return run_small(h, d_phase, B, d_frames, d_slopes, st);
    }
    int F, ks;
    schedule(h, B, &F, &ks);
    int rc = ensure_scratch(h, F, ks, st, true);
    if (rc) return rc;
    const size_t NN = (size_t)t.N * t.N, DD = (size_t)t.D * t.D, SS = (size_t)2 * t.n_valid;
    const size_t n_chunks = ((size_t)B + F - 1) / F;
    if (n_chunks == 1) {                       // a single chunk (closed loop): everything in order on the caller's stream
        if ((rc = launch_k1(h, d_phase, B, st))) return rc;
        if ((rc = launch_k2(h, B, ks, st))) return rc;
        return launch_tail(h, B, d_frames, d_slopes, ks, st);
    }
    // several chunks: the small, latency-bound tail kernels of chunk c run on a side stream under the row pass of
    // chunk c+1; the column pass of chunk c+1 waits for them (they read colbin), the caller's stream joins at the end
    if (!h->out_stream) PWFS_CUDA(h, cudaStreamCreateWithFlags(&h->out_stream, cudaStreamNonBlocking));
    if ((rc = ensure_chunk_events(h, n_chunks))) return rc;
    size_t c = 0;
    for (int f0 = 0; f0 < B; f0 += F, ++c) {
        const int Fc = std::min(F, B - f0);
        if ((rc = launch_k1(h, d_phase + (size_t)f0 * NN, Fc, st))) return rc;
        if (c > 0) PWFS_CUDA(h, cudaStreamWaitEvent(st, h->tail_ev[c - 1], 0));
        if ((rc = launch_k2(h, Fc, ks, st))) return rc;
        PWFS_CUDA(h, cudaEventRecord(h->done_ev[c], st));
        PWFS_CUDA(h, cudaStreamWaitEvent(h->out_stream, h->done_ev[c], 0));
        if ((rc = launch_tail(h, Fc, d_frames + (size_t)f0 * DD, d_slopes ? d_slopes + (size_t)f0 * SS : nullptr, ks, h->out_stream)))
            return rc;
        PWFS_CUDA(h, cudaEventRecord(h->tail_ev[c], h->out_stream));
    }
    PWFS_CUDA(h, cudaStreamWaitEvent(st, h->tail_ev[n_chunks - 1], 0));
    return PWFS_OK;
}

int pwfs_debug_intensity(pwfs_t *h, const float *d_phase, int32_t B, float *d_intensity, void *cuda_stream) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_phase || !d_intensity) return PWFS_EINVAL;
    DeviceGuard dg(h->device);
    PWFS_CUDA(h, dg.err);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DevTables &t = h->tab;
    const size_t NN = (size_t)t.N * t.N, MM = (size_t)t.M * t.M;
    // one frame at a time, the whole modulation loop in one warp (k_split 1) so that dbg holds the complete sum
    int rc = ensure_scratch(h, 1, 1, st, true);
    if (rc) return rc;
    float *dbg = nullptr;
    PWFS_CUDA(h, cudaMalloc((void **)&dbg, (size_t)t.ncols * t.M * sizeof(float)));
    const double m4 = h->quarter ? std::pow((double)t.M, 4.0) : 1.0;
    const int o = t.M / 2 - t.N / 2;                                  // O2: the oracle's pupil sits at [o, o + N)
    cudaError_t e = cudaMemsetAsync(d_intensity, 0, (size_t)B * MM * sizeof(float), st);
    for (int b = 0; b < B && e == cudaSuccess && !rc; ++b) {
        t.dbg_I = dbg;
        rc = launch_k1(h, d_phase + (size_t)b * NN, 1, st);
        if (!rc) rc = launch_k2(h, 1, 1, st);
        t.dbg_I = nullptr;
        if (!rc) {
            debug_scatter_kernel<<<dim3(t.ncols, 1), 256, 0, st>>>(t, dbg, d_intensity + (size_t)b * MM, o,
                                                                   (float)(1.0 / ((double)t.K * m4)));
            rc = check_launch(h, 2);
        }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);               // test-only: synchronous, then free the buffer
    cudaFree(dbg);
    if (e != cudaSuccess) { h->last_cuda = (int)e; return PWFS_ECUDA; }
    return rc;
}

int pwfs_run_host(pwfs_t *h, const float *h_phase, int32_t B, float *h_frames, float *h_slopes) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!h_phase || !h_frames || h->debug_only) return PWFS_EINVAL;
    DeviceGuard dg(h->device);
    PWFS_CUDA(h, dg.err);
    const DevTables &t = h->tab;
    const size_t NN = (size_t)t.N * t.N, DD = (size_t)t.D * t.D, SS = (size_t)2 * t.n_valid;
    if (!h->hstream) PWFS_CUDA(h, cudaStreamCreateWithFlags(&h->hstream, cudaStreamNonBlocking));
    if ((size_t)B > h->d_cap_frames) {
        if (h->d_phase) cudaFree(h->d_phase);
        if (h->d_frames) cudaFree(h->d_frames);
        if (h->d_slopes) cudaFree(h->d_slopes);
        h->d_phase = h->d_frames = h->d_slopes = nullptr; h->d_cap_frames = 0;
        cudaError_t e = cudaMalloc((void **)&h->d_phase, (size_t)B * NN * sizeof(float));
        if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_frames, (size_t)B * DD * sizeof(float));
        if (e == cudaSuccess) e = cudaMalloc((void **)&h->d_slopes, (size_t)B * SS * sizeof(float));
        if (e != cudaSuccess) { h->last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? PWFS_ENOMEM : PWFS_ECUDA; }
        h->d_cap_frames = (size_t)B;
    }
    if (small_applies(h, B)) {                                     // one fused launch between the two copies
        int rc = ensure_small(h, B, h->hstream, false);
        if (rc) return rc;
        PWFS_CUDA(h, cudaMemcpyAsync(h->d_phase, h_phase, (size_t)B * NN * sizeof(float), cudaMemcpyHostToDevice, h->hstream));
        if ((rc = run_small(h, h->d_phase, B, h->d_frames, h_slopes ? h->d_slopes : nullptr, h->hstream))) return rc;
        PWFS_CUDA(h, cudaMemcpyAsync(h_frames, h->d_frames, (size_t)B * DD * sizeof(float), cudaMemcpyDeviceToHost, h->hstream));
        if (h_slopes)
            PWFS_CUDA(h, cudaMemcpyAsync(h_slopes, h->d_slopes, (size_t)B * SS * sizeof(float), cudaMemcpyDeviceToHost, h->hstream));
        PWFS_CUDA(h, cudaStreamSynchronize(h->hstream));
        return PWFS_OK;
    }
    if (!h->in_stream) PWFS_CUDA(h, cudaStreamCreateWithFlags(&h->in_stream, cudaStreamNonBlocking));
    if (!h->out_stream) PWFS_CUDA(h, cudaStreamCreateWithFlags(&h->out_stream, cudaStreamNonBlocking));
    int F, ks;
    // a short first chunk (the only copy-in nothing can hide), then three large ones (few partly filled last waves)
    int first = (h->user_fpc <= 0 && B >= 16) ? std::max(1, B / 16) : 0;
    schedule(h, B - first, &F, &ks, first ? 3 : 1);              // small batches: one chunk, copies are short anyway
    first = std::min(first, F);                                  // scratch (and grid.z) hold F frames, the short chunk too
    int rc = ensure_scratch(h, F, ks);
    if (rc) return rc;
    const size_t n_chunks = (first ? 1 : 0) + ((size_t)(B - first) + F - 1) / F;
    if ((rc = ensure_chunk_events(h, n_chunks))) return rc;
    // three streams, chunk by chunk: the copy-in of chunk c+1, and the tail kernels and the copy-out of chunk c-1,
    // run under the FFT kernels of chunk c (pinned host memory; pageable memory degrades to staged copies)
    size_t c = 0;
    for (int f0 = 0, Fc = 0; f0 < B; f0 += Fc, ++c) {
        Fc = (c == 0 && first) ? first : std::min(F, B - f0);
        float *dp = h->d_phase + (size_t)f0 * NN, *df = h->d_frames + (size_t)f0 * DD, *ds = h->d_slopes + (size_t)f0 * SS;
        PWFS_CUDA(h, cudaMemcpyAsync(dp, h_phase + (size_t)f0 * NN, (size_t)Fc * NN * sizeof(float), cudaMemcpyHostToDevice, h->in_stream));
        PWFS_CUDA(h, cudaEventRecord(h->in_ev[c], h->in_stream));
        PWFS_CUDA(h, cudaStreamWaitEvent(h->hstream, h->in_ev[c], 0));
        if ((rc = launch_k1(h, dp, Fc, h->hstream))) return rc;
        if (c > 0) PWFS_CUDA(h, cudaStreamWaitEvent(h->hstream, h->tail_ev[c - 1], 0));   // colbin is free again
        if ((rc = launch_k2(h, Fc, ks, h->hstream))) return rc;
        PWFS_CUDA(h, cudaEventRecord(h->done_ev[c], h->hstream));
        PWFS_CUDA(h, cudaStreamWaitEvent(h->out_stream, h->done_ev[c], 0));
        if ((rc = launch_tail(h, Fc, df, h_slopes ? ds : nullptr, ks, h->out_stream))) return rc;
        PWFS_CUDA(h, cudaEventRecord(h->tail_ev[c], h->out_stream));
        PWFS_CUDA(h, cudaMemcpyAsync(h_frames + (size_t)f0 * DD, df, (size_t)Fc * DD * sizeof(float), cudaMemcpyDeviceToHost, h->out_stream));
        if (h_slopes)
            PWFS_CUDA(h, cudaMemcpyAsync(h_slopes + (size_t)f0 * SS, ds, (size_t)Fc * SS * sizeof(float), cudaMemcpyDeviceToHost, h->out_stream));
    }
    PWFS_CUDA(h, cudaStreamSynchronize(h->out_stream));
    PWFS_CUDA(h, cudaStreamSynchronize(h->hstream));
    return PWFS_OK;
}

// pwfs_run for callers that cannot allocate (include/pwfs.h has the contract).  Same fused kernel as pwfs_run's
// small-batch path on the M = 128 grid, same arguments; the only difference is where the kernel's working memory
// lives.  Nothing here calls cudaMalloc / cudaFree, creates a stream or an event, or touches the handle's own scratch.
int pwfs_run_noalloc(pwfs_t *h, const float *d_phase, int32_t B, float *d_frames, float *d_slopes, void *cuda_stream) {
    if (!h || B < 0) return PWFS_EINVAL;
    if (B == 0) return PWFS_OK;
    if (!d_phase || !d_frames || h->debug_only) return PWFS_EINVAL;
    const DevTables &t = h->tab;
    // geometry the fused kernel's shared-memory plan holds (SmallCfg::MAXN, MAXCOLS, MAXD, MAXCMAX)
    if (!h->L.launch_s || t.N > 64 || t.ncols > 128 || t.D > 64 || t.cmax > 8) return PWFS_EUNSUPPORTED;
    const size_t DD = (size_t)t.D * t.D;
    if (B > kNoAllocFrames || (size_t)B * t.K * DD > kNoAllocPartFloats) return PWFS_ELIMIT;
    DeviceGuard dg(h->device);
    PWFS_CUDA(h, dg.err);
    unsigned char *base = nullptr;
    PWFS_CUDA(h, noalloc_scratch_address(h->device, &base));      // first call on this GPU: looks the array up
    unsigned *counter = reinterpret_cast<unsigned *>(base);
    float *part = reinterpret_cast<float *>(base + kNoAllocCounterBytes);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The array keeps whatever the previous call (of any handle) left.  The partial frames are fully overwritten before
    // they are read; the counters must be zero when the kernel starts, and a call that was cut short could have left
    // them otherwise -- so they are cleared in stream order, every time.
    PWFS_CUDA(h, cudaMemsetAsync(counter, 0, (size_t)B * sizeof(unsigned), st));
    const double m4 = h->quarter ? std::pow((double)t.M, 4.0) : 1.0;
    h->launches[4]++;
    h->L.launch_s(dim3(t.K, B), st, t, d_phase, part, counter, d_frames, d_slopes, (float)(1.0 / ((double)t.K * m4)));
    return check_launch(h, 4);
}

}  // extern "C"
