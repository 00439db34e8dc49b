// lisatdi.cu -- the C ABI of include/lisatdi.h: argument checks, tile plan, launches.
// Single translation unit: the kernels live in orbit.cuh and response.cuh.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "common.cuh"
#include "orbit.cuh"
#include "response.cuh"
#include "fast.cuh"

namespace {

std::atomic<int64_t> g_launches{0};
inline void count_launch(int k = 1) { g_launches.fetch_add(k, std::memory_order_relaxed); }

/* Per-kernel timing (ltdi_profile_*): while enabled, every kernel launch is bracketed by two CUDA events on
 * the stream it is launched on; ltdi_profile_read() turns the pairs into per-kernel totals. */
struct ProfPair { int id; cudaEvent_t e0, e1; };
std::mutex g_prof_mu;
bool g_prof_on = false;
std::vector<ProfPair> g_prof_pending;
std::vector<cudaEvent_t> g_prof_pool;
double g_prof_ms[3 * LTDI_KERNEL_COUNT] = {};   /* [which][kernel] */
int64_t g_prof_n[3 * LTDI_KERNEL_COUNT] = {};

struct ProfScope {
    cudaStream_t st;
    ProfPair pr;
    bool on;
    static cudaEvent_t get()
    {
        cudaEvent_t e = nullptr;
        if (!g_prof_pool.empty()) { e = g_prof_pool.back(); g_prof_pool.pop_back(); }
        else if (cudaEventCreate(&e) != cudaSuccess) { (void)cudaGetLastError(); e = nullptr; }
        return e;
    }
    ProfScope(int id, cudaStream_t s) : st(s), on(false)
    {
        std::lock_guard<std::mutex> lk(g_prof_mu);
        if (!g_prof_on) return;
        pr.id = id; pr.e0 = get(); pr.e1 = get();
        if (pr.e0 && pr.e1) { on = true; cudaEventRecord(pr.e0, st); }
    }
    ~ProfScope()
    {
        if (!on) return;
        cudaEventRecord(pr.e1, st);
        std::lock_guard<std::mutex> lk(g_prof_mu);
        g_prof_pending.push_back(pr);
    }
};

// Per-device state.  __constant__ tables, cudaFuncSetAttribute, streams and events all belong to ONE device: a
// process that uses several devices gets one DeviceState per device (indexed by cudaGetDevice()).
#define LTDI_HOST_CHUNKS 16   /* most pieces an end-to-end call is cut into */
struct DeviceState {
    std::mutex mu;                 /* guards everything below, and serialises the hybrid fork / join on the device */
    bool ready = false;
    int status = LTDI_OK;
    int smem_max = 0, sms = 0;
    cudaStream_t side = nullptr;   /* non-blocking side stream of the hybrid's concurrent launches */
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    /* ltdi_response_host: copy streams and the events that chain upload -> kernels -> download chunk by chunk */
    std::mutex host_mu;
    cudaStream_t copy_in = nullptr, copy_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_done = nullptr, ev_in[LTDI_HOST_CHUNKS] = {}, ev_comp[LTDI_HOST_CHUNKS] = {};
    std::vector<std::pair<const void *, size_t>> smem_seen;   /* cudaFuncAttributeMaxDynamicSharedMemorySize per kernel */
};
DeviceState g_dev[64];

// 1 / prod_{m != k}(k - m), k, m = -(M/2-1) .. M/2, for every even M <= 64 (rows of c_lag_inv_den), and the
// scale factors of the symmetric pair form, uploaded to the CURRENT device
int upload_constants()
{
    int status = LTDI_OK;
    {
        std::vector<double> tab(32 * LTDI_MAX_TAPS, 0.0);
        for (int r = 0; r < 32; ++r) {
            const int M = 2 * (r + 1), kmin = -(M / 2 - 1);
            for (int i = 0; i < M; ++i) {
                long double den = 1.0L;
                for (int j = 0; j < M; ++j)
                    if (j != i) den *= (long double)((kmin + i) - (kmin + j));
                tab[r * LTDI_MAX_TAPS + i] = (double)(1.0L / den);
            }
        }
        if (cudaMemcpyToSymbol(c_lag_inv_den, tab.data(), tab.size() * sizeof(double)) != cudaSuccess) {
            (void)cudaGetLastError();
            status = LTDI_ECUDA;
        }
        /* symmetric pair form (fast.cuh): lambda_i with prod_{i != j} lambda_i = c_j = 1 / (2 a_j prod_{i != j}
         * (a_j^2 - a_i^2)), a_j = j + 1/2.  With Lambda = prod lambda_i: lambda_j = Lambda / c_j and
         * Lambda^(H-1) = prod c_i; computed through logarithms in long double (prod c_i underflows). */
        double lam[2][16] = {}, kap[2][16] = {};
        const int Hs[2] = {5, 16};
        for (int r = 0; r < 2; ++r) {
            const int H = Hs[r];
            long double c[16], logsum = 0.0L;
            int neg = 0;
            for (int j = 0; j < H; ++j) {
                const long double aj = j + 0.5L;
                long double den = 2.0L * aj;
                for (int i = 0; i < H; ++i)
                    if (i != j) den *= aj * aj - (i + 0.5L) * (i + 0.5L);
                c[j] = 1.0L / den;
                logsum += logl(fabsl(c[j]));
                neg += c[j] < 0;
            }
            /* sign: H - 1 odd -> Lambda takes the sign of prod c_i; H - 1 even -> prod c_i > 0 for H = 5 */
            long double Lambda = expl(logsum / (H - 1));
            if (((H - 1) & 1) && (neg & 1)) Lambda = -Lambda;
            for (int j = 0; j < H; ++j) {
                const long double l = Lambda / c[j];
                lam[r][j] = (double)l;
                kap[r][j] = (double)(-l * (j + 0.5L) * (j + 0.5L));
            }
        }
        if (cudaMemcpyToSymbol(c_sym_lam, lam, sizeof lam) != cudaSuccess ||
            cudaMemcpyToSymbol(c_sym_kap, kap, sizeof kap) != cudaSuccess) {
            (void)cudaGetLastError();
            status = LTDI_ECUDA;
        }
    }
    return status;
}

/* the state of the current device, initialised on first use */
int device_state(DeviceState **out)
{
    int dev = 0;
    LTDI_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return LTDI_EUNSUPPORTED;
    DeviceState &d = g_dev[dev];
    std::lock_guard<std::mutex> lk(d.mu);
    if (!d.ready) {
        d.status = upload_constants();
        if (d.status == LTDI_OK) {
            if (cudaDeviceGetAttribute(&d.smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess ||
                cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
                cudaStreamCreateWithFlags(&d.side, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&d.ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&d.ev_join, cudaEventDisableTiming) != cudaSuccess ||
                cudaStreamCreateWithFlags(&d.copy_in, cudaStreamNonBlocking) != cudaSuccess ||
                cudaStreamCreateWithFlags(&d.copy_out, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&d.ev_start, cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&d.ev_done, cudaEventDisableTiming) != cudaSuccess) {
                (void)cudaGetLastError();
                d.status = LTDI_ECUDA;
            }
            for (int i = 0; i < LTDI_HOST_CHUNKS && d.status == LTDI_OK; ++i)
                if (cudaEventCreateWithFlags(&d.ev_in[i], cudaEventDisableTiming) != cudaSuccess ||
                    cudaEventCreateWithFlags(&d.ev_comp[i], cudaEventDisableTiming) != cudaSuccess) {
                    (void)cudaGetLastError();
                    d.status = LTDI_ECUDA;
                }
        }
        d.ready = true;
    }
    *out = &d;
    return d.status;
}

int64_t iceil(double x) { return (int64_t)std::ceil(x); }

// G11 / O10: closed-form reaches.  Projection: |k.R|/c + L <= 1.02 (R + arm)/c plus half a stencil;
// TDI: 7 light times (gen 2.0) or 3 (gen 1.5) backwards with a 3 % allowance, plus half a stencil.
Margins compute_margins(const ltdi_orbit_desc &d, int gen, int order, int fd_order)
{
    Margins m;
    const int M = order + 1;
    m.m1 = iceil(1.02 * (d.R_m + d.arm_m) / LTDI_C_LIGHT / d.dt) + M / 2;
    m.m2 = iceil((gen == LTDI_GEN_20 ? 7.2 : 3.1) * (d.arm_m / LTDI_C_LIGHT) / d.dt) + M / 2;
    m.w = fd_order / 2;
    m.lo = m.m1 + m.m2 + 2 * m.w;
    m.hi = m.m1 + M / 2 + 2 * m.w;
    return m;
}

bool desc_ok(const ltdi_orbit_desc *d)
{
    return d && d->n > 0 && d->dt > 0.0 && d->arm_m > 0.0 && d->R_m > 0.0 && d->period_s > 0.0 &&
           d->mode >= LTDI_ORBIT_STATIC_EQUALARM && d->mode <= LTDI_ORBIT_KNOTS;
}
bool order_ok(int order) { return order >= 1 && order <= 63 && (order & 1); }
bool gen_ok(int gen) { return gen == LTDI_GEN_15 || gen == LTDI_GEN_20; }

int64_t table_stride(int64_t n) { return (n + 31) / 32 * 32; }

struct KnotGrid { int64_t nk; double t0, dt; int order; };

int orbits_common(const ltdi_orbit_desc *desc, const double *d_R, const double *d_L, void *d_tables, size_t bytes,
                  void *stream, ltdi_orbits **out, const KnotGrid *kg = nullptr)
{
    if (!desc_ok(desc) || !d_tables || !out) return LTDI_EINVAL;
    const int64_t stride = table_stride(desc->n);
    if (bytes < (size_t)stride * LTDI_TABLE_BYTES_PER_SAMPLE) return LTDI_EWORKSPACE;
    if ((uintptr_t)d_tables % 16) return LTDI_EINVAL;
    OrbitKernelParams p;
    std::memset(&p, 0, sizeof p);
    p.t0 = desc->t0; p.dt = desc->dt; p.n = desc->n; p.stride = stride;
    p.arm_m = desc->arm_m; p.R_m = desc->R_m;
    /* constants of the launch in long double, handed to the kernel as double-double pairs */
    auto split = [](long double v) { dd r; r.hi = (double)v; r.lo = (double)(v - (long double)r.hi); return r; };
    const long double pi_l = 3.14159265358979323846264338327950288L;
    const long double omega_l = 2.0L * pi_l / (long double)desc->period_s;
    p.omega = (double)omega_l; p.omega_dd = split(omega_l);
    p.alpha0 = desc->alpha0; p.mode = desc->mode;
    long double sb_l[3], cb_l[3];
    for (int i = 0; i < 3; ++i) { /* beta_i = 2 pi (i - 1) / 3 + rot0 */
        const long double beta = 2.0L * pi_l * (long double)i / 3.0L + (long double)desc->rot0;
        sb_l[i] = sinl(beta); cb_l[i] = cosl(beta);
        p.sb[i] = split(sb_l[i]); p.cb[i] = split(cb_l[i]);
    }
    {
        const long double L = desc->arm_m, R = desc->R_m;
        const long double e = L / (2.0L * sqrtl(3.0L) * R);
        p.half_eR = split(0.5L * e * R);
        p.s3_eR = split(sqrtl(3.0L) * e * R);
        p.inv_c = split(1.0L / (long double)LTDI_C_LIGHT);
        p.L_static = split(L / (long double)LTDI_C_LIGHT);
        for (int l = 0; l < 3; ++l) {   /* unit vectors of the rigid triangle: coefficients with 1 / L folded in */
            const int s = link_sender(l), r = link_receiver(l);
            const long double dc = cb_l[r] - cb_l[s], dsn = sb_l[r] - sb_l[s];
            p.PA[l] = split(0.5L * e * R * dc / L); p.PB[l] = split(0.5L * e * R * dsn / L);
            p.PA3[l] = split(1.5L * e * R * dc / L); p.PB3[l] = split(1.5L * e * R * dsn / L);
            p.PC[l] = split(sqrtl(3.0L) * e * R * dc / L); p.PD[l] = split(sqrtl(3.0L) * e * R * dsn / L);
        }
        long double f = 1.0L;   /* (-1)^m / (2m+1)! and (-1)^m / (2m)! */
        for (int m = 0; m < 12; ++m) {
            if (m > 0) f *= (long double)(2 * m - 1) * (long double)(2 * m);
            p.cos_c[m] = split(((m & 1) ? -1.0L : 1.0L) / f);
            if (m < 11) p.sin_c[m] = split(((m & 1) ? -1.0L : 1.0L) / (f * (long double)(2 * m + 1)));
        }
    }
    p.R_in = d_R; p.L_in = d_L; p.tab = (double *)d_tables;
    if (kg) {
        p.nk = kg->nk; p.tk0 = kg->t0; p.dtk = kg->dt; p.korder = kg->order;
        p.inv_dtk = split(1.0L / (long double)kg->dt);
        DeviceState *ds = nullptr;   /* the knot weights read the Lagrange denominators of the device */
        const int rc = device_state(&ds);
        if (rc) return rc;
    }
    const int threads = 128;
    const int64_t blocks = (desc->n + threads - 1) / threads;
    {
        ProfScope ps(LTDI_KERNEL_ORBIT, (cudaStream_t)stream);
        if (kg) orbit_delay_kernel<true><<<(unsigned)blocks, threads, 0, (cudaStream_t)stream>>>(p);
        else orbit_delay_kernel<false><<<(unsigned)blocks, threads, 0, (cudaStream_t)stream>>>(p);
    }
    count_launch();
    LTDI_CUDA_OK(cudaGetLastError());
    ltdi_orbits *o = new (std::nothrow) ltdi_orbits;
    if (!o) return LTDI_EINVAL;
    o->desc = *desc;
    o->d_tab = (const double *)d_tables;
    o->stride = stride;
    o->d_anc = nullptr;
    o->anc_gen = 0;
    o->anc_M = 0;
    o->anc_has2 = false;
    *out = o;
    return LTDI_OK;
}

// workspace layout (doubles): raw sources [batch][3] | frames [batch][16] | hybrid windows [n_hyb][4] | hybrid tile
// plan [batch][4] (eight 32-bit integers per source, HybPlan) | waveform model constants [batch][20] (ChirpDev, 8(f)-3)
size_t work_doubles(int64_t batch) { return ((size_t)batch * (3 + LTDI_FRAME_STRIDE + 4 + 4 + LTDI_CHIRP_STRIDE) + 31) / 32 * 32; }

bool fast_order(int order) { return order == 9 || order == 31; }

/* workspace of the fast path behind the per-source parameters: anchors | anchor headers | link-series scratch
 * for one chunk of sources | (hybrid) the compact tile lists of the chunk.  Chunks of up to 2 GiB of scratch: measured
 * on B200, large chunks (fewer launches, fewer grid tails) beat chunks small enough to keep the link series in the
 * 126 MB L2 (96 MB: 5 % slower at cfg4s) -- the scratch traffic, 96 B per sample, is < 5 % of the HBM bandwidth at the
 * speed of these FP64-bound kernels. */
struct FastLayout {
    int64_t ntilesA, ntilesAL, ntilesC, ntilesN, lds, chunk;   /* link tiles (full, LFA), TDI tiles, anchor tiles (= 448-sample blocks) */
    size_t anc, hdr, anc2, y, lists;     /* doubles */
    size_t total;                  /* doubles, including work_doubles(batch) */
};
FastLayout fast_layout(int which, int64_t n, int64_t batch, int M, bool want_y = true)
{
    FastLayout f;
    f.ntilesA = (n + FAST_TA - 1) / FAST_TA;
    f.ntilesAL = (n + FAST_TAL - 1) / FAST_TAL;
    f.ntilesC = (n + tdi_tc(which) - 1) / tdi_tc(which);
    f.ntilesN = (n + FAST_TCA - 1) / FAST_TCA;
    f.lds = (n + 15) / 16 * 16;
    /* rows of link scratch per source: six full links, three derivatives of the LFA links + the three LFA links themselves
     * (written only when the caller asks for d_y) */
    const int rows = which == LTDI_RESPONSE_FULL ? 6 : which == LTDI_RESPONSE_LFA ? 6 : 12;
    const int rows_noy = which == LTDI_RESPONSE_FULL ? 6 : which == LTDI_RESPONSE_LFA ? 3 : 9;   /* without d_y */
    const size_t cap = (size_t)2048 << 20; /* bytes of scratch per chunk */
    int64_t chunk = (int64_t)(cap / ((size_t)rows * f.lds * sizeof(double)));
    f.chunk = chunk < 1 ? 1 : (chunk > batch ? batch : chunk);
    /* the memory is sized for a call that returns the links; a call that does not fits more sources into the same scratch */
    const int64_t chunk_noy = std::min<int64_t>(batch, (int64_t)(((size_t)rows * f.chunk) / rows_noy));
    const int64_t chunk_y = f.chunk;
    f.anc = (size_t)f.ntilesN * FAST_NA * FAST_ANC_DOUBLES(M);
    f.hdr = (size_t)f.ntilesN * FAST_NA * 4;
    f.anc2 = (size_t)f.ntilesN * FAST_NA * M;   /* second derivative of the weights (second-order instances) */
    f.y = (size_t)rows * chunk_y * f.lds;
    /* hybrid: link tiles of both kinds, LFA-only blocks, blend blocks, full-only 224-sample tiles (int2 each) */
    f.lists = which == LTDI_RESPONSE_HYBRID ? (size_t)chunk_noy * (f.ntilesA + f.ntilesAL + 4 * f.ntilesN) : 0;
    if (!want_y) f.chunk = chunk_noy;
    f.total = work_doubles(batch) + f.anc + f.hdr + f.anc2 + f.y + f.lists;
    return f;
}

// ---- hybrid tile plan (S8) ---------------------------------------------------------------------------------------
// Per source the host classifies the 448-sample blocks from (t_hyb, T): blocks [0, nLt) lie entirely before the
// window (w_Full = 0 on every sample, with one sample of margin: LFA only), blocks [fFt, nblk) entirely after it
// (w_LFA = 0: full response only), blocks [nLt, fFt) need both and the blend of Eq. (4.6).  Everything else -- which
// link tiles are needed, how many CTAs every launch has -- follows from these two integers by the integer rules of
// hyb_counts(), evaluated identically on the host (grid sizes, list offsets) and in hybrid_plan_kernel (list entries).
struct HybPlan { int nLt, fFt, off_link_full, off_link_lfa, off_lfa, off_blend, off_full, pad; };
struct HybGeom { int64_t n, ntilesA, nblk; int back, fwd; };
struct HybCounts { int64_t lfa_link, full_link_first, full_link, lfa_blk, blend_blk, full_first, full_tiles; };
__host__ __device__ inline HybCounts hyb_counts(const HybGeom &g, int nLt, int fFt)
{
    HybCounts c;
    /* LFA links: read by the TDI stage of blocks [0, fFt), up to `fwd` samples past their end */
    int64_t endL = fFt == 0 ? 0 : (int64_t)fFt * FAST_TCA + g.fwd;
    if (endL > g.n) endL = g.n;
    c.lfa_link = (endL + FAST_TAL - 1) / FAST_TAL;   /* LFA link tiles store the derivative of FAST_TAL samples */
    /* full links: read by the TDI stage of blocks [nLt, nblk), from `back` samples before their start */
    int64_t first = (int64_t)nLt * FAST_TCA - g.back;
    if (first < 0) first = 0;
    c.full_link_first = nLt >= g.nblk ? g.ntilesA : first / FAST_TA;
    c.full_link = g.ntilesA - c.full_link_first;
    c.lfa_blk = nLt;
    c.blend_blk = fFt - nLt;
    c.full_first = 2 * (int64_t)fFt;   /* 224-sample tiles of the FULL instance */
    c.full_tiles = fFt >= g.nblk ? 0 : (g.n - (int64_t)fFt * FAST_TCA + tdi_tc(LTDI_RESPONSE_FULL) - 1) / tdi_tc(LTDI_RESPONSE_FULL);
    return c;
}
static_assert(FAST_TCA == 2 * tdi_tc(LTDI_RESPONSE_FULL) && FAST_TCA == tdi_tc(LTDI_RESPONSE_HYBRID) && FAST_TCA == tdi_tc(LTDI_RESPONSE_LFA),
              "the hybrid plan counts 448-sample blocks");

struct PlanArgs {
    HybGeom g;
    const HybPlan *plan;      /* [nb] of the chunk (device), or nullptr: `small` */
    HybPlan small[32];
    int64_t b0, nb;
    int2 *link_list, *lfa_list, *blend_list, *full_list;
    int64_t n_link_full;      /* LFA-link items follow the full-link items in link_list */
};

/* blockIdx.y = source of the chunk, threads over the tile slot j: writes the (source, tile) entries of the five lists.
 * Heavy tiles first: the full-link items precede the LFA-link items, and late (full) tiles precede early ones. */
__global__ void hybrid_plan_kernel(const __grid_constant__ PlanArgs a)
{
    const int64_t b = blockIdx.y;
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const HybPlan pl = a.plan ? a.plan[b] : a.small[a.b0 + b];
    const HybCounts c = hyb_counts(a.g, pl.nLt, pl.fFt);
    if (j < c.full_link) a.link_list[pl.off_link_full + j] = make_int2((int)b, (int)(a.g.ntilesA - 1 - j));
    if (j < c.lfa_link) a.link_list[a.n_link_full + pl.off_link_lfa + j] = make_int2((int)b, (int)j);
    if (j < c.lfa_blk) a.lfa_list[pl.off_lfa + j] = make_int2((int)b, (int)j);
    if (j < c.blend_blk) a.blend_list[pl.off_blend + j] = make_int2((int)b, (int)(pl.nLt + j));
    if (j < c.full_tiles) a.full_list[pl.off_full + j] = make_int2((int)b, (int)(c.full_first + j));
}

/* nLt, fFt of one source (host): block k = samples [448 k, min(448 (k + 1), n)), one sample of margin on either side
 * so that the per-sample weights of the kernels (their own fp64 rounding of t_n) can never disagree with the class */
void classify_blocks(const ltdi_orbit_desc &d, const ltdi_hybrid &h, int64_t nblk, int *nLt, int *fFt)
{
    auto lfa_only = [&](int64_t k) {
        const int64_t e = std::min((k + 1) * (int64_t)FAST_TCA, d.n) - 1;
        return d.t0 + (double)e * d.dt + d.dt - h.t_hyb < -0.5 * h.window_s;
    };
    auto full_only = [&](int64_t k) { return d.t0 + (double)(k * FAST_TCA) * d.dt - d.dt - h.t_hyb > 0.5 * h.window_s; };
    auto guess = [&](double t) {
        const double k = std::floor((t - d.t0) / d.dt / (double)FAST_TCA);
        return (int64_t)std::min(std::max(k, 0.0), (double)nblk);
    };
    int64_t a = guess(h.t_hyb - 0.5 * h.window_s);
    while (a < nblk && lfa_only(a)) ++a;
    while (a > 0 && !lfa_only(a - 1)) --a;
    int64_t f = guess(h.t_hyb + 0.5 * h.window_s);
    while (f > 0 && full_only(f - 1)) --f;
    while (f < nblk && !full_only(f)) ++f;
    if (f < a) f = a;
    *nLt = (int)a;
    *fFt = (int)f;
}

struct SmallArgs { double v[32 * 7]; }; /* batch <= 32: sources and windows travel as kernel arguments */

__global__ void unpack_small_kernel(SmallArgs a, int batch, int n_hyb, double *src, double *frames, HybDev *hyb)
{
    const int i = threadIdx.x;
    if (i < batch * 3) src[i] = a.v[i];
    if (i < n_hyb * 4) ((double *)hyb)[i] = a.v[96 + i];
    if (i < batch) source_frame_one(a.v[3 * i], a.v[3 * i + 1], a.v[3 * i + 2], frames + i * LTDI_FRAME_STRIDE); /* S1 */
}

/* batch > 32: the parameters of up to 512 sources per launch travel as kernel arguments (28 KB; CUDA >= 12.1 allows
 * 32 764 bytes on sm_70+).  A cudaMemcpyAsync from pageable host memory above 64 KB would block the host until the
 * stream has drained, which leaves the GPU idle between the calls of a step. */
#define LTDI_BIG_SOURCES 256
struct BigArgs { double src[LTDI_BIG_SOURCES * 3]; double hyb[LTDI_BIG_SOURCES * 4]; HybPlan plan[LTDI_BIG_SOURCES]; };

__global__ void unpack_big_kernel(const __grid_constant__ BigArgs a, int count, int n_hyb_here, int n_plan, double *src,
                                  double *frames, double *hyb, HybPlan *plan)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) {
        src[3 * i] = a.src[3 * i]; src[3 * i + 1] = a.src[3 * i + 1]; src[3 * i + 2] = a.src[3 * i + 2];
        source_frame_one(a.src[3 * i], a.src[3 * i + 1], a.src[3 * i + 2], frames + i * LTDI_FRAME_STRIDE); /* S1 */
    }
    if (i < n_hyb_here) {
        hyb[4 * i] = a.hyb[4 * i]; hyb[4 * i + 1] = a.hyb[4 * i + 1];
        hyb[4 * i + 2] = a.hyb[4 * i + 2]; hyb[4 * i + 3] = a.hyb[4 * i + 3];
    }
    if (i < n_plan) plan[i] = a.plan[i];
}

template <typename K>
int set_smem(DeviceState &ds, K kernel, size_t smem)
{
    if (smem > (size_t)ds.smem_max) return LTDI_EUNSUPPORTED;
    if (smem + 4096 <= 48 * 1024) return LTDI_OK;   /* the kernels' static shared memory (<= 2 KB) counts too */
    /* the attribute is sticky per device function and device: raise it only when a call needs more than any before */
    std::lock_guard<std::mutex> lk(ds.mu);
    for (auto &e : ds.smem_seen)
        if (e.first == (const void *)kernel) {
            if (e.second >= smem) return LTDI_OK;
            LTDI_CUDA_OK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            e.second = smem;
            return LTDI_OK;
        }
    LTDI_CUDA_OK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ds.smem_seen.emplace_back((const void *)kernel, smem);
    return LTDI_OK;
}

template <int MT, bool STAGE>
int launch_response(DeviceState &ds, const RespParams &p, int threads, size_t smem, cudaStream_t st)
{
    const int rc = set_smem(ds, response_kernel<MT, STAGE>, smem);
    if (rc) return rc;
    {
        ProfScope ps(LTDI_KERNEL_GENERIC + LTDI_KERNEL_COUNT * p.which, st);
        response_kernel<MT, STAGE><<<(unsigned)(p.ntiles * p.batch), threads, smem, st>>>(p);
    }
    count_launch();
    LTDI_CUDA_OK(cudaGetLastError());
    return LTDI_OK;
}

/* waveform model constants of `batch` sources to the device: kernel arguments in slices of 96 sources (as BigArgs) */
#define LTDI_CHIRP_SLICE 96
struct ChirpArgs { ChirpDev v[LTDI_CHIRP_SLICE]; };
__global__ void unpack_chirp_kernel(const __grid_constant__ ChirpArgs a, int count, ChirpDev *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count * LTDI_CHIRP_STRIDE) reinterpret_cast<double *>(out)[i] = reinterpret_cast<const double *>(a.v)[i];
}
int upload_chirps(const ltdi_chirp *h_wav, int64_t batch, double t0, ChirpDev *d_out, cudaStream_t st)
{
    ChirpArgs *a = new (std::nothrow) ChirpArgs;
    if (!a) return LTDI_EINVAL;
    for (int64_t b0 = 0; b0 < batch; b0 += LTDI_CHIRP_SLICE) {
        const int cnt = (int)std::min<int64_t>(LTDI_CHIRP_SLICE, batch - b0);
        for (int i = 0; i < cnt; ++i)
            if (chirp_fill(h_wav[b0 + i], t0, &a->v[i])) { delete a; return LTDI_EINVAL; }
        unpack_chirp_kernel<<<(cnt * LTDI_CHIRP_STRIDE + 127) / 128, 128, 0, st>>>(*a, cnt, d_out + b0);
        count_launch();
        if (cudaGetLastError() != cudaSuccess) { delete a; return LTDI_ECUDA; }
    }
    delete a;
    return LTDI_OK;
}

/* constants of the eccentric model of `batch` sources to the device, as kernel arguments in slices */
#define LTDI_ECC_SLICE 256
struct EccArgs { EccDev v[LTDI_ECC_SLICE]; };
__global__ void unpack_ecc_kernel(const __grid_constant__ EccArgs a, int count, EccDev *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count * LTDI_ECC_STRIDE) reinterpret_cast<double *>(out)[i] = reinterpret_cast<const double *>(a.v)[i];
}

/* host side of the hybrid plan: per-source plans (offsets relative to the source's chunk) and per-chunk totals */
struct ChunkTotals { int64_t link_full, link_lfa, lfa, blend, full, max_slots; };
struct HybHost {
    std::vector<HybPlan> plan;        /* [batch] */
    std::vector<ChunkTotals> chunk;   /* [number of chunks] */
    HybGeom g;
};

int build_hybrid_plan(const ltdi_orbit_desc &d, const Margins &mg, int M, const FastLayout &lay, int64_t batch,
                      const ltdi_hybrid *h_hyb, int64_t n_hyb, HybHost *out)
{
    out->g.n = d.n; out->g.ntilesA = lay.ntilesA; out->g.nblk = lay.ntilesN;
    out->g.back = tdi_back(mg.m2) + 2;
    out->g.fwd = M / 2 + 4 + 2 * (int)mg.w;
    out->plan.resize((size_t)batch);
    out->chunk.clear();
    int nLt = 0, fFt = 0;
    for (int64_t b0 = 0; b0 < batch; b0 += lay.chunk) {
        const int64_t nb = std::min(lay.chunk, batch - b0);
        ChunkTotals t = {0, 0, 0, 0, 0, 0};
        for (int64_t b = b0; b < b0 + nb; ++b) {
            if (n_hyb != 1 || b == 0) classify_blocks(d, h_hyb[n_hyb == 1 ? 0 : b], lay.ntilesN, &nLt, &fFt);
            const HybCounts c = hyb_counts(out->g, nLt, fFt);
            if (std::max({t.link_full + c.full_link, t.link_lfa + c.lfa_link, t.lfa + c.lfa_blk, t.blend + c.blend_blk,
                          t.full + c.full_tiles}) >= ((int64_t)1 << 31))
                return LTDI_EUNSUPPORTED;
            HybPlan &pl = out->plan[(size_t)b];
            pl.nLt = nLt; pl.fFt = fFt; pl.pad = 0;
            pl.off_link_full = (int)t.link_full; pl.off_link_lfa = (int)t.link_lfa; pl.off_lfa = (int)t.lfa;
            pl.off_blend = (int)t.blend; pl.off_full = (int)t.full;
            t.link_full += c.full_link; t.link_lfa += c.lfa_link; t.lfa += c.lfa_blk; t.blend += c.blend_blk;
            t.full += c.full_tiles;
            t.max_slots = std::max({t.max_slots, c.full_link, c.lfa_link, c.lfa_blk, c.blend_blk, c.full_tiles});
        }
        out->chunk.push_back(t);
    }
    return LTDI_OK;
}

/* the first-order (analytic orbits) or second-order (tables, numerical orbits, nested delays) instance of the TDI kernel */
template <int M, int WHICH>
void launch_tdi(bool ord2, unsigned grid, size_t smem, cudaStream_t st, const FastParams &p)
{
    if (ord2) tdi_kernel<M, WHICH, true><<<grid, tdi_threads(WHICH), smem, st>>>(p);
    else tdi_kernel<M, WHICH, false><<<grid, tdi_threads(WHICH), smem, st>>>(p);
}
template <int M, int WHICH>
int set_smem_tdi(DeviceState &ds, bool ord2, size_t smem)
{
    return ord2 ? set_smem(ds, tdi_kernel<M, WHICH, true>, smem) : set_smem(ds, tdi_kernel<M, WHICH, false>, smem);
}

// the tuned path: anchors once per call, then link kernel(s) and TDI kernel(s) per chunk of sources
template <int M>
int run_fast(DeviceState &ds, const RespParams &rp, const Margins &mg, const ltdi_orbits *orb, int which, double *work,
             cudaStream_t st, const double *small /* [32 * 7] host values or nullptr */, const HybHost *hh,
             const HybPlan *d_plan /* [batch] device copies of hh->plan, or nullptr when small */)
{
    constexpr int H = M / 2;
    const ltdi_orbit_desc &d = orb->desc;
    const FastLayout lay = fast_layout(which, d.n, rp.batch, M, rp.Y != nullptr);
    if (mg.m2 > 4096 || mg.m1 > 8192) return LTDI_EUNSUPPORTED;

    FastParams p;
    std::memset(&p, 0, sizeof p);
    p.tab = rp.tab; p.stride = rp.stride; p.n = rp.n; p.t0 = rp.t0; p.dt = rp.dt; p.inv_dt = 1.0 / rp.dt;
    p.ld = rp.ld; p.n_hyb = rp.n_hyb; p.which = which; p.gen = rp.gen; p.fd = rp.fd;
    p.m1 = mg.m1; p.m2 = mg.m2; p.w = mg.w; p.lo = mg.lo; p.hi = mg.hi; p.qmax = rp.qmax;
    p.lfa_terms = rp.lfa_terms; p.lfa_point = rp.lfa_point; p.xw = rp.xw;
    p.inv_fd3 = 1.0 / ((mg.w == 1 ? 2.0 : 8.0) * rp.dt * rp.dt * rp.dt);
    p.m2_15 = compute_margins(d, LTDI_GEN_15, M - 1, 0).m2;
    p.m2_20 = compute_margins(d, LTDI_GEN_20, M - 1, 0).m2;
    p.inv_fd1 = 1.0 / ((mg.w == 1 ? 2.0 : 12.0) * rp.dt);
    p.inv_fd2 = 1.0 / ((mg.w == 1 ? 1.0 : 12.0) * rp.dt * rp.dt);
    p.lds = lay.lds; p.batch_all = rp.batch; p.ntilesA = lay.ntilesA; p.ntilesC = lay.ntilesC;
    p.use_small = small != nullptr;
    if (small) {
        std::memcpy(p.small, small, sizeof p.small);
        for (int64_t b = 0; b < rp.batch && b < 32; ++b) {   /* S1 on the host, Eq. (2.1) with G1 and (2.3), in long double */
            const long double be = small[3 * b], la = small[3 * b + 1], ps = small[3 * b + 2];
            const long double sb = sinl(be), cb = cosl(be), sl = sinl(la), cl = cosl(la);
            double *f = p.small_fr + 11 * b;
            f[0] = (double)(-cb * cl); f[1] = (double)(-cb * sl); f[2] = (double)(-sb);   /* k = -e_r */
            f[3] = (double)sl;         f[4] = (double)(-cl);      f[5] = 0.0;             /* u = -e_phi */
            f[6] = (double)(-sb * cl); f[7] = (double)(-sb * sl); f[8] = (double)cb;      /* v = -e_theta */
            f[9] = (double)cosl(2.0L * ps); f[10] = (double)sinl(2.0L * ps);
        }
    }
    double *anc = work, *hdr = anc + lay.anc, *anc2 = hdr + lay.hdr, *ys = anc2 + lay.anc2;
    int2 *lists = reinterpret_cast<int2 *>(ys + lay.y);
    p.anc = anc; p.anc_hdr = hdr;
    /* second-order weights where the light times of the orbit object may drift by more than FAST_DMAX over a tile
     * (caller's tables, numerical orbit files) and for nested delays; the analytic orbits keep the first-order instances */
    const bool ord2 = d.mode == LTDI_ORBIT_TABLES || d.mode == LTDI_ORBIT_KNOTS || rp.nested;
    p.anc2 = ord2 ? anc2 : nullptr; p.nested = rp.nested;

    const bool full = which != LTDI_RESPONSE_LFA, lfa = which != LTDI_RESPONSE_FULL;
    const bool hybrid = which == LTDI_RESPONSE_HYBRID;
    /* staged strain (4 parity-split series) + the orbit-table rows of the tile */
    const size_t smem_strain = (size_t)4 * ((FAST_TA + 2 * mg.m1 + 4) / 2) * sizeof(double);
    const size_t smem_link = smem_strain + (size_t)LTDI_TABLE_ROWS * FAST_TA * sizeof(double);
    const size_t smem_link_lfa = smem_strain + (size_t)(ROW_L + 3) * FAST_TA * sizeof(double) +
                                 (size_t)lfa_raw_doubles((int)((FAST_TA + 2 * mg.m1 + 4) / 2)) * sizeof(double) +          /* + raw strain */
                                 (size_t)LFA_LO_ROWS * LFA_TLW * sizeof(float) +                          /* + low parts */
                                 (rp.lfa_terms >= 2 ? smem_strain : 0);                                     /* + d^3h/dt^3 numerators */
    const size_t smem_link_hyb = std::max(smem_link, smem_link_lfa);
    const size_t smem_tdi_full = tdi_smem_bytes<M>(LTDI_RESPONSE_FULL, mg.m2, mg.w, ord2);
    const size_t smem_tdi_hyb = tdi_smem_bytes<M>(LTDI_RESPONSE_HYBRID, mg.m2, mg.w, ord2);
    const size_t smem_tdi_lfa = tdi_smem_bytes<M>(LTDI_RESPONSE_LFA, mg.m2, mg.w, ord2);
    int rc;
    if (hybrid) {
        if ((rc = set_smem(ds, link_hybrid_kernel<H>, smem_link_hyb))) return rc;
        if ((rc = set_smem_tdi<M, LTDI_RESPONSE_HYBRID>(ds, ord2, smem_tdi_hyb))) return rc;
    } else {
        if (full && (rc = set_smem(ds, link_kernel<H, false>, smem_link))) return rc;
        if (lfa && (rc = set_smem(ds, link_kernel<H, true>, smem_link_lfa))) return rc;
    }
    if (full && (rc = set_smem_tdi<M, LTDI_RESPONSE_FULL>(ds, ord2, smem_tdi_full))) return rc;
    if (lfa && (rc = set_smem_tdi<M, LTDI_RESPONSE_LFA>(ds, ord2, smem_tdi_lfa))) return rc;

    if (orb->d_anc && orb->anc_M == M && (!ord2 || orb->anc_has2)) {
        /* ltdi_orbits_prepare() has computed the anchors of this order for the time grid (they serve both generations) */
        p.anc = orb->d_anc;
        p.anc_hdr = orb->d_anc + lay.anc;
        p.anc2 = ord2 ? orb->d_anc + lay.anc + lay.hdr : nullptr;
    } else {
        ProfScope ps(LTDI_KERNEL_ANCHOR + LTDI_KERNEL_COUNT * which, st);
        anchor_kernel<M><<<(unsigned)lay.ntilesN, 64, 0, st>>>(p, anc, hdr, ord2 ? anc2 : nullptr);
        count_launch();
        LTDI_CUDA_OK(cudaGetLastError());
    }

    /* the hybrid forks its LFA blocks onto the device's side stream: one call at a time per device uses the events */
    std::unique_lock<std::mutex> fork_lock(ds.mu, std::defer_lock);
    if (hybrid) fork_lock.lock();

    int64_t ichunk = 0;
    for (int64_t b0 = 0; b0 < rp.batch; b0 += lay.chunk, ++ichunk) {
        const int64_t nb = std::min(lay.chunk, rp.batch - b0);
        p.batch = nb; p.b0 = b0;
        p.hp = rp.hp + b0 * rp.ld; p.hc = rp.hc + b0 * rp.ld;
        p.frames = rp.frames + b0 * LTDI_FRAME_STRIDE;
        p.hyb = (const double *)rp.hyb + (rp.n_hyb == 1 ? 0 : 4 * b0);
        p.A = rp.A + b0 * rp.ld; p.E = rp.E + b0 * rp.ld; p.T = rp.T + b0 * rp.ld;
        p.XYZ = rp.XYZ; p.Y = rp.Y;
        p.yF = ys; p.yL = ys + (full ? (size_t)6 * nb * lay.lds : 0);
        p.yLraw = (lfa && rp.Y) ? p.yL + (size_t)3 * nb * lay.lds : nullptr;
        p.work = nullptr; p.nwork = 0; p.nwork_full = 0;
        if (lay.ntilesAL * nb >= ((int64_t)1 << 31) || lay.ntilesC * nb >= ((int64_t)1 << 31)) return LTDI_EUNSUPPORTED;
        if (!hybrid) {
            if (full) {
                {
                    ProfScope ps(LTDI_KERNEL_LINK_FULL + LTDI_KERNEL_COUNT * which, st);
                    if (rp.chirp) link_chirp_kernel<<<(unsigned)(lay.ntilesA * nb), FAST_TA_THREADS, 0, st>>>(p, rp.chirp + b0);
                    else link_kernel<H, false><<<(unsigned)(lay.ntilesA * nb), FAST_TA_THREADS, smem_link, st>>>(p);
                }
                count_launch();
                ProfScope ps(LTDI_KERNEL_TDI + LTDI_KERNEL_COUNT * which, st);
                launch_tdi<M, LTDI_RESPONSE_FULL>(ord2, (unsigned)(lay.ntilesC * nb), smem_tdi_full, st, p);
            } else {
                {
                    ProfScope ps(LTDI_KERNEL_LINK_LFA + LTDI_KERNEL_COUNT * which, st);
                    link_kernel<H, true><<<(unsigned)(lay.ntilesAL * nb), FAST_TA_THREADS, smem_link_lfa, st>>>(p);
                }
                count_launch();
                p.nwork = lay.ntilesN * nb;
                ProfScope ps(LTDI_KERNEL_TDI_LFA + LTDI_KERNEL_COUNT * which, st);
                launch_tdi<M, LTDI_RESPONSE_LFA>(ord2, (unsigned)p.nwork, smem_tdi_lfa, st, p);
            }
            count_launch();
            LTDI_CUDA_OK(cudaGetLastError());
            continue;
        }

        /* hybrid: compact lists, then one launch per class of tiles */
        const ChunkTotals &ct = hh->chunk[(size_t)ichunk];
        int2 *l_link = lists, *l_lfa = l_link + (size_t)nb * (lay.ntilesA + lay.ntilesAL), *l_blend = l_lfa + (size_t)nb * lay.ntilesN,
             *l_full = l_blend + (size_t)nb * lay.ntilesN;
        {
            PlanArgs a;
            std::memset(&a, 0, sizeof a);
            a.g = hh->g;
            a.plan = d_plan ? d_plan + b0 : nullptr;
            if (!d_plan) std::memcpy(a.small, hh->plan.data(), hh->plan.size() * sizeof(HybPlan));
            a.b0 = b0; a.nb = nb;
            a.link_list = l_link; a.lfa_list = l_lfa; a.blend_list = l_blend; a.full_list = l_full;
            a.n_link_full = ct.link_full;
            if (ct.max_slots > 0) {
                ProfScope ps(LTDI_KERNEL_PLAN + LTDI_KERNEL_COUNT * which, st);
                hybrid_plan_kernel<<<dim3((unsigned)((ct.max_slots + 127) / 128), (unsigned)nb), 128, 0, st>>>(a);
                count_launch();
            }
        }
        if (ct.link_full + ct.link_lfa > 0) {
            p.work = l_link; p.nwork = ct.link_full + ct.link_lfa; p.nwork_full = ct.link_full;
            ProfScope ps(LTDI_KERNEL_LINK_FULL + LTDI_KERNEL_COUNT * which, st);
            link_hybrid_kernel<H><<<(unsigned)p.nwork, FAST_TA_THREADS, smem_link_hyb, st>>>(p);
            count_launch();
        }
        const bool side_lfa = ct.lfa > 0 && (ct.blend > 0 || ct.full > 0);   /* concurrent launches only if both exist */
        if (ct.lfa > 0) {
            cudaStream_t s_lfa = st;
            if (side_lfa) {   /* fork: the LFA blocks on the side stream, beside the blend and full-only tiles */
                LTDI_CUDA_OK(cudaEventRecord(ds.ev_fork, st));
                LTDI_CUDA_OK(cudaStreamWaitEvent(ds.side, ds.ev_fork, 0));
                s_lfa = ds.side;
            }
            p.work = l_lfa; p.nwork = ct.lfa; p.nwork_full = 0;
            {
                ProfScope ps(LTDI_KERNEL_TDI_LFA + LTDI_KERNEL_COUNT * which, s_lfa);
                launch_tdi<M, LTDI_RESPONSE_LFA>(ord2, (unsigned)p.nwork, smem_tdi_lfa, s_lfa, p);
            }
            count_launch();
            if (side_lfa) LTDI_CUDA_OK(cudaEventRecord(ds.ev_join, ds.side));
        }
        {
            ProfScope ps(LTDI_KERNEL_TDI + LTDI_KERNEL_COUNT * which, st);
            if (ct.full > 0) {
                p.work = l_full; p.nwork = ct.full;
                launch_tdi<M, LTDI_RESPONSE_FULL>(ord2, (unsigned)ct.full, smem_tdi_full, st, p);
                count_launch();
            }
            if (ct.blend > 0) {
                p.work = l_blend; p.nwork = ct.blend;
                launch_tdi<M, LTDI_RESPONSE_HYBRID>(ord2, (unsigned)ct.blend, smem_tdi_hyb, st, p);
                count_launch();
            }
        }
        if (side_lfa) LTDI_CUDA_OK(cudaStreamWaitEvent(st, ds.ev_join, 0));   /* join before the scratch is reused */
        LTDI_CUDA_OK(cudaGetLastError());
    }
    return LTDI_OK;
}

int run_response(int which, const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                 int64_t batch, const ltdi_source *h_src, int gen, int order, int fd_order,
                 const ltdi_hybrid *h_hyb, int64_t n_hyb, double *d_A, double *d_E, double *d_T, double *d_XYZ,
                 double *d_y, void *d_work, size_t work_bytes, void *stream, int lfa_terms = 1,
                 int lfa_point = LTDI_LFA_CENTRAL, int nested_order = 0, const ltdi_chirp *h_wav = nullptr, int lfa6 = 0,
                 int sagnac = 0)
{
    if (sagnac && (which != LTDI_RESPONSE_FULL || nested_order != 0 || h_wav)) return LTDI_EINVAL;
    if (lfa6 && (which != LTDI_RESPONSE_LFA || lfa_terms != 1 || lfa_point != LTDI_LFA_CENTRAL)) return LTDI_EINVAL;
    if (nested_order != 0 && (which != LTDI_RESPONSE_FULL || nested_order != 3)) return nested_order == 3 || nested_order < 0 || !(nested_order & 1) ? LTDI_EINVAL : LTDI_EUNSUPPORTED;
    if (nested_order && !fast_order(order)) return LTDI_EUNSUPPORTED;   /* nested delays run on the tuned path (orders 9, 31) */
    if (lfa_terms < 1 || lfa_terms > 2 || lfa_point < LTDI_LFA_CENTRAL || lfa_point > LTDI_LFA_FORWARD) return LTDI_EINVAL;
    if (lfa_terms == 2 && lfa_point != LTDI_LFA_CENTRAL) return LTDI_EINVAL;
    if ((lfa_terms != 1 || lfa_point != LTDI_LFA_CENTRAL) && which != LTDI_RESPONSE_LFA) return LTDI_EINVAL;
    if (!orb || ((!d_hp || !d_hc) && !h_wav) || !h_src || !d_A || !d_E || !d_T || !d_work) return LTDI_EINVAL;
    if (h_wav && (which != LTDI_RESPONSE_FULL || !fast_order(order))) return which != LTDI_RESPONSE_FULL ? LTDI_EINVAL : LTDI_EUNSUPPORTED;
    if (!gen_ok(gen) || !order_ok(order) || batch < 1 || ld < orb->desc.n) return LTDI_EINVAL;
    if (which != LTDI_RESPONSE_FULL && fd_order != 2 && fd_order != 4) return LTDI_EINVAL;
    if (which == LTDI_RESPONSE_FULL) fd_order = 0;
    if (which == LTDI_RESPONSE_HYBRID) {
        if (!h_hyb || (n_hyb != 1 && n_hyb != batch)) return LTDI_EINVAL;
        for (int64_t i = 0; i < n_hyb; ++i) {
            if (h_hyb[i].taper != LTDI_TAPER_SIGMOID && h_hyb[i].taper != LTDI_TAPER_COSINE) return LTDI_EINVAL;
            if (!(h_hyb[i].window_s > 0.0)) return LTDI_EINVAL;
            if (h_hyb[i].taper == LTDI_TAPER_SIGMOID && !(h_hyb[i].sigma_s > 0.0)) return LTDI_EINVAL;
        }
    } else {
        n_hyb = 0;
    }
    if ((uintptr_t)d_work % 16) return LTDI_EINVAL;
    {
        const size_t need = fast_order(order) ? fast_layout(which, orb->desc.n, batch, order + 1).total : work_doubles(batch);
        if (work_bytes < need * sizeof(double)) return LTDI_EWORKSPACE;
    }
    if (batch * ((orb->desc.n + 63) / 64) >= (int64_t)1 << 31) return LTDI_EUNSUPPORTED;
    DeviceState *dsp = nullptr;
    int rc = device_state(&dsp);
    if (rc) return rc;
    DeviceState &ds = *dsp;
    cudaStream_t st = (cudaStream_t)stream;
    const ltdi_orbit_desc &d = orb->desc;
    Margins mg = compute_margins(d, gen, order, fd_order);
    /* the third-derivative stencil is one sample wider than the first ((B4) m = 1 term: of the strain; (B30): of the links) */
    const int xw = (lfa_terms >= 2 || (lfa6 && gen == LTDI_GEN_20)) ? 1 : 0;
    mg.lo += xw; mg.hi += xw;
    const int M = order + 1;

    /* hybrid on the tuned path: the tile plan (host integers; see classify_blocks / hyb_counts) */
    HybHost hh;
    const bool plan_hybrid = which == LTDI_RESPONSE_HYBRID && fast_order(order) && mg.m2 <= 4096 && mg.m1 <= 8192;
    if (plan_hybrid) {
        rc = build_hybrid_plan(d, mg, M, fast_layout(which, d.n, batch, M, d_y != nullptr), batch, h_hyb, n_hyb, &hh);
        if (rc) return rc;
    }

    /* S1: per-source parameters to the device, then the source-frame kernel */
    double *w_src = (double *)d_work;
    double *w_frames = w_src + 3 * batch;
    HybDev *w_hyb = (HybDev *)(w_frames + LTDI_FRAME_STRIDE * batch);
    HybPlan *w_plan = (HybPlan *)((double *)w_hyb + 4 * batch);
    ChirpDev *w_chirp = (ChirpDev *)((double *)w_plan + 4 * batch);
    if (h_wav) {   /* the model constants of every source (host, long double) to the workspace */
        const int rcw = upload_chirps(h_wav, batch, orb->desc.t0, w_chirp, st);
        if (rcw) return rcw;
    }
    SmallArgs small_args;
    bool have_small = false;   /* batch <= 32: the tuned kernels take the parameters as arguments (no launch) */
    if (batch <= 32) {
        SmallArgs a;
        std::memset(&a, 0, sizeof a);
        for (int64_t b = 0; b < batch; ++b) {
            a.v[3 * b + 0] = h_src[b].beta; a.v[3 * b + 1] = h_src[b].lambda; a.v[3 * b + 2] = h_src[b].psi;
        }
        for (int64_t i = 0; i < n_hyb; ++i) {
            a.v[96 + 4 * i + 0] = h_hyb[i].t_hyb; a.v[96 + 4 * i + 1] = h_hyb[i].window_s;
            a.v[96 + 4 * i + 2] = h_hyb[i].sigma_s; a.v[96 + 4 * i + 3] = (double)h_hyb[i].taper;
        }
        small_args = a;
        have_small = true;
    } else {
        BigArgs *big = new (std::nothrow) BigArgs;
        if (!big) return LTDI_EINVAL;
        for (int64_t b0 = 0; b0 < batch; b0 += LTDI_BIG_SOURCES) {
            const int cnt = (int)std::min<int64_t>(LTDI_BIG_SOURCES, batch - b0);
            for (int i = 0; i < cnt; ++i) {
                big->src[3 * i + 0] = h_src[b0 + i].beta; big->src[3 * i + 1] = h_src[b0 + i].lambda;
                big->src[3 * i + 2] = h_src[b0 + i].psi;
            }
            int nh = 0;   /* hybrid windows of this slice (n_hyb is 0, 1 or batch) */
            if (n_hyb == batch) nh = cnt;
            else if (n_hyb == 1 && b0 == 0) nh = 1;
            for (int i = 0; i < nh; ++i) {
                const ltdi_hybrid &h = h_hyb[n_hyb == 1 ? 0 : b0 + i];
                big->hyb[4 * i + 0] = h.t_hyb; big->hyb[4 * i + 1] = h.window_s;
                big->hyb[4 * i + 2] = h.sigma_s; big->hyb[4 * i + 3] = (double)h.taper;
            }
            if (plan_hybrid) std::memcpy(big->plan, hh.plan.data() + b0, (size_t)cnt * sizeof(HybPlan));
            {
                ProfScope ps(LTDI_KERNEL_PREP + LTDI_KERNEL_COUNT * which, st);
                unpack_big_kernel<<<(LTDI_BIG_SOURCES + 127) / 128, 128, 0, st>>>(
                    *big, cnt, nh, plan_hybrid ? cnt : 0, w_src + 3 * b0, w_frames + LTDI_FRAME_STRIDE * b0,
                    (double *)w_hyb + (n_hyb == 1 ? 0 : 4 * b0), w_plan + b0);
            }
            count_launch();
            if (cudaGetLastError() != cudaSuccess) { delete big; return LTDI_ECUDA; }
        }
        delete big;   /* kernel arguments are copied at launch */
    }

    /* tile plan */
    RespParams p;
    std::memset(&p, 0, sizeof p);
    p.tab = orb->d_tab; p.stride = orb->stride; p.n = d.n; p.t0 = d.t0; p.dt = d.dt;
    p.hp = d_hp; p.hc = d_hc; p.ld = ld; p.batch = batch;
    p.frames = w_frames; p.hyb = w_hyb; p.n_hyb = n_hyb;
    p.which = which; p.gen = gen; p.M = M; p.fd = fd_order;
    p.m1 = mg.m1; p.m2 = mg.m2; p.w = mg.w; p.lo = mg.lo; p.hi = mg.hi;
    p.qmax = (int)(mg.m1 - M / 2);
    p.lfa_terms = lfa_terms; p.lfa_point = lfa_point; p.xw = xw; p.nested = nested_order != 0;
    p.chirp = h_wav ? w_chirp : nullptr;
    p.lfa6 = lfa6;
    p.sagnac = sagnac;
    p.A = d_A; p.E = d_E; p.T = d_T; p.XYZ = d_XYZ; p.Y = d_y;

    if (fast_order(order) && !lfa6 && !sagnac) {   /* (B20) / (B30) and the Sagnac combinations run on the generic kernel for every order */
        const double *sm = have_small ? small_args.v : nullptr;
        const HybPlan *dp = have_small ? nullptr : w_plan;
        double *fw = (double *)d_work + work_doubles(batch);
        const int frc = M == 32 ? run_fast<32>(ds, p, mg, orb, which, fw, st, sm, &hh, dp)
                                : run_fast<10>(ds, p, mg, orb, which, fw, st, sm, &hh, dp);
        if (frc != LTDI_EUNSUPPORTED || nested_order) return frc;   /* else: shapes the tuned kernels do not cover */
    }
    if (have_small) { /* the generic kernel reads frames and windows from the workspace */
        {
            ProfScope ps(LTDI_KERNEL_PREP + LTDI_KERNEL_COUNT * which, st);
            unpack_small_kernel<<<1, 128, 0, st>>>(small_args, (int)batch, (int)n_hyb, w_src, w_frames, w_hyb);
        }
        count_launch();
        LTDI_CUDA_OK(cudaGetLastError());
    }

    int tile = 256;
    while (tile > 64 && ((d.n + tile - 1) / tile) * batch < 2 * 148) tile /= 2; /* fill the 148 SMs */
    const int smem_max = ds.smem_max;
    bool stage = true;
    size_t smem = 0;
    for (;;) {
        p.tile = tile;
        p.yr = (int)(tile + mg.m2 + M / 2 + 1);
        p.hw = (int)(p.yr + 2 * mg.m1 + 6 * mg.w + 2 + 2 * xw);
        const int w = (int)mg.w;
        size_t off = 0;
        if (which != LTDI_RESPONSE_LFA) off += 6 * (size_t)p.yr;
        p.off_yL = (int)off;
        if (which != LTDI_RESPONSE_FULL) off += lfa6 ? 6 * (size_t)(p.yr + 2 * (w + xw)) : 3 * (size_t)(p.yr + 2 * w);
        p.off_dL = (int)off;
        if (which != LTDI_RESPONSE_FULL) off += (lfa6 ? 12 : 3) * (size_t)p.yr;
        p.off_hs = (int)off;
        if (stage) off += 2 * (size_t)p.hw;
        smem = off * sizeof(double);
        if (smem <= (size_t)smem_max) break;
        if (stage) { stage = false; continue; }      /* very small dt: read the strain through L1 instead */
        if (tile > 64) { tile /= 2; continue; }
        return LTDI_EUNSUPPORTED;
    }
    p.ntiles = (d.n + tile - 1) / tile;
    const int threads = tile >= 256 ? 256 : 128;
    if (M == 32)
        return stage ? launch_response<32, true>(ds, p, threads, smem, st) : launch_response<32, false>(ds, p, threads, smem, st);
    if (M == 10)
        return stage ? launch_response<10, true>(ds, p, threads, smem, st) : launch_response<10, false>(ds, p, threads, smem, st);
    return stage ? launch_response<0, true>(ds, p, threads, smem, st) : launch_response<0, false>(ds, p, threads, smem, st);
}

// register-resident DFMA chains: the FP64 pipe's issue rate, used as the "alu" roofline peak
__global__ void __launch_bounds__(256) fp64_probe_kernel(double *out, int iters)
{
    double a[8];
    const double x = 1.0 + 1e-9 * (double)threadIdx.x, y = 1e-12 * (double)(blockIdx.x + 1);
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = (double)i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = fma(a[i], x, y);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

} // namespace

extern "C" {

int ltdi_fp64_probe(double *d_out, int blocks, int iters, void *stream, double *dfma_per_launch)
{
    if (!d_out || blocks < 1 || iters < 1) return LTDI_EINVAL;
    fp64_probe_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(d_out, iters);
    count_launch();
    LTDI_CUDA_OK(cudaGetLastError());
    if (dfma_per_launch) *dfma_per_launch = (double)blocks * 256.0 * 64.0 * (double)iters;
    return LTDI_OK;
}

int ltdi_host_scratch_bytes(int64_t ld, int64_t batch, size_t *bytes)
{
    if (ld < 1 || batch < 1 || !bytes) return LTDI_EINVAL;
    const size_t series = ((size_t)ld * (size_t)batch * sizeof(double) + 255) / 256 * 256;
    size_t work = 0; /* the chunking of the link scratch differs per response: size for the largest */
    for (int which = LTDI_RESPONSE_FULL; which <= LTDI_RESPONSE_HYBRID; ++which)
        work = std::max(work, fast_layout(which, ld, batch, 32).total);
    *bytes = 5 * series + (work * sizeof(double) + 255) / 256 * 256;
    return LTDI_OK;
}

int ltdi_response_host(int which, const ltdi_orbits *orb, const double *h_hp, const double *h_hc, int64_t ld,
                       int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, int fd_order,
                       const ltdi_hybrid *h_hyb, int64_t n_hyb, double *h_A, double *h_E, double *h_T,
                       void *d_scratch, size_t scratch_bytes, void *stream)
{
    if (!h_hp || !h_hc || !h_A || !h_E || !h_T || !d_scratch || ld < 1 || batch < 1) return LTDI_EINVAL;
    if (which < LTDI_RESPONSE_FULL || which > LTDI_RESPONSE_HYBRID) return LTDI_EINVAL;
    if ((uintptr_t)d_scratch % 256) return LTDI_EINVAL;
    size_t need = 0;
    ltdi_host_scratch_bytes(ld, batch, &need);
    if (scratch_bytes < need) return LTDI_EWORKSPACE;
    const size_t bytes = (size_t)ld * (size_t)batch * sizeof(double);
    const size_t series = (bytes + 255) / 256 * 256;
    char *base = (char *)d_scratch;
    double *d_hp = (double *)base, *d_hc = (double *)(base + series);
    double *d_A = (double *)(base + 2 * series), *d_E = (double *)(base + 3 * series), *d_T = (double *)(base + 4 * series);
    void *d_work = base + 5 * series;
    cudaStream_t st = (cudaStream_t)stream;
    /* A large batch is cut into pieces of whole sources that go through upload -> kernels -> download as a pipeline: the
     * uploads on one copy stream, the kernels on the caller's stream, the downloads on a second copy stream, chained by
     * events, so that a single call keeps both directions of PCIe and the SMs busy at once.  The caller's stream waits
     * for the last download: the results are valid once `stream` has been synchronised, as for a one-piece call. */
    const int64_t piece_min = std::max<int64_t>(1, ((int64_t)64 << 20) / (ld * (int64_t)sizeof(double)));   /* >= 64 MiB per series */
    const int npiece = (int)std::max<int64_t>(1, std::min<int64_t>(LTDI_HOST_CHUNKS, batch / piece_min));
    if (npiece == 1) {
        LTDI_CUDA_OK(cudaMemcpyAsync(d_hp, h_hp, bytes, cudaMemcpyHostToDevice, st));
        LTDI_CUDA_OK(cudaMemcpyAsync(d_hc, h_hc, bytes, cudaMemcpyHostToDevice, st));
        const int rc = run_response(which, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, fd_order, h_hyb,
                                    n_hyb, d_A, d_E, d_T, nullptr, nullptr, d_work, need - 5 * series, stream);
        if (rc) return rc;
        LTDI_CUDA_OK(cudaMemcpyAsync(h_A, d_A, bytes, cudaMemcpyDeviceToHost, st));
        LTDI_CUDA_OK(cudaMemcpyAsync(h_E, d_E, bytes, cudaMemcpyDeviceToHost, st));
        LTDI_CUDA_OK(cudaMemcpyAsync(h_T, d_T, bytes, cudaMemcpyDeviceToHost, st));
        return LTDI_OK;
    }
    if (!h_src || (which == LTDI_RESPONSE_HYBRID && (!h_hyb || (n_hyb != 1 && n_hyb != batch)))) return LTDI_EINVAL;
    DeviceState *dsp = nullptr;
    int rc = device_state(&dsp);
    if (rc) return rc;
    DeviceState &ds = *dsp;
    std::lock_guard<std::mutex> lk(ds.host_mu);   /* one call at a time issues into the copy streams and their events */
    LTDI_CUDA_OK(cudaEventRecord(ds.ev_start, st));
    LTDI_CUDA_OK(cudaStreamWaitEvent(ds.copy_in, ds.ev_start, 0));    /* what the caller queued before this call comes first */
    LTDI_CUDA_OK(cudaStreamWaitEvent(ds.copy_out, ds.ev_start, 0));
    const int64_t per = (batch + npiece - 1) / npiece;
    int used = 0;
    for (int c = 0; c < npiece; ++c) {
        const int64_t b0 = c * per, cnt = std::min(per, batch - b0);
        if (cnt <= 0) break;
        const size_t off = (size_t)b0 * (size_t)ld, nb = (size_t)cnt * (size_t)ld * sizeof(double);
        LTDI_CUDA_OK(cudaMemcpyAsync(d_hp + off, h_hp + off, nb, cudaMemcpyHostToDevice, ds.copy_in));
        LTDI_CUDA_OK(cudaMemcpyAsync(d_hc + off, h_hc + off, nb, cudaMemcpyHostToDevice, ds.copy_in));
        LTDI_CUDA_OK(cudaEventRecord(ds.ev_in[c], ds.copy_in));
        LTDI_CUDA_OK(cudaStreamWaitEvent(st, ds.ev_in[c], 0));
        rc = run_response(which, orb, d_hp + off, d_hc + off, ld, cnt, h_src + b0, gen, lagrange_order, fd_order,
                          h_hyb ? h_hyb + (n_hyb == batch ? b0 : 0) : nullptr, n_hyb == batch ? cnt : n_hyb, d_A + off,
                          d_E + off, d_T + off, nullptr, nullptr, d_work, need - 5 * series, stream);
        if (rc) break;
        LTDI_CUDA_OK(cudaEventRecord(ds.ev_comp[c], st));
        LTDI_CUDA_OK(cudaStreamWaitEvent(ds.copy_out, ds.ev_comp[c], 0));
        LTDI_CUDA_OK(cudaMemcpyAsync(h_A + off, d_A + off, nb, cudaMemcpyDeviceToHost, ds.copy_out));
        LTDI_CUDA_OK(cudaMemcpyAsync(h_E + off, d_E + off, nb, cudaMemcpyDeviceToHost, ds.copy_out));
        LTDI_CUDA_OK(cudaMemcpyAsync(h_T + off, d_T + off, nb, cudaMemcpyDeviceToHost, ds.copy_out));
        ++used;
    }
    /* also after an error: the caller's stream must not run ahead of copies that were already queued */
    (void)used;
    LTDI_CUDA_OK(cudaEventRecord(ds.ev_done, ds.copy_out));
    LTDI_CUDA_OK(cudaStreamWaitEvent(st, ds.ev_done, 0));
    LTDI_CUDA_OK(cudaEventRecord(ds.ev_done, ds.copy_in));
    LTDI_CUDA_OK(cudaStreamWaitEvent(st, ds.ev_done, 0));
    return rc;
}

int ltdi_orbits_workspace_bytes(const ltdi_orbit_desc *desc, size_t *bytes)
{
    if (!desc_ok(desc) || !bytes) return LTDI_EINVAL;
    *bytes = (size_t)table_stride(desc->n) * LTDI_TABLE_BYTES_PER_SAMPLE;
    return LTDI_OK;
}

int ltdi_orbits_init(const ltdi_orbit_desc *desc, void *d_tables, size_t bytes, void *stream, ltdi_orbits **out)
{
    if (desc && (desc->mode == LTDI_ORBIT_TABLES || desc->mode == LTDI_ORBIT_KNOTS)) return LTDI_EINVAL;
    return orbits_common(desc, nullptr, nullptr, d_tables, bytes, stream, out);
}

int ltdi_orbits_init_knots(const ltdi_orbit_desc *desc, const double *d_knots, int64_t nk, double knot_t0, double knot_dt,
                           int knot_order, void *d_tables, size_t bytes, void *stream, ltdi_orbits **out)
{
    if (!desc_ok(desc) || desc->mode != LTDI_ORBIT_KNOTS || !d_knots) return LTDI_EINVAL;
    if (knot_order < 1 || knot_order > 15 || !(knot_order & 1) || !(knot_dt > 0.0) || nk < knot_order + 1) return LTDI_EINVAL;
    const int M = knot_order + 1;
    const double t_end = desc->t0 + (double)(desc->n - 1) * desc->dt;
    if (knot_t0 + (double)(M / 2 - 1) * knot_dt > desc->t0 || t_end > knot_t0 + (double)(nk - 1 - M / 2) * knot_dt) return LTDI_EINVAL;
    const KnotGrid kg = {nk, knot_t0, knot_dt, knot_order};
    return orbits_common(desc, d_knots, nullptr, d_tables, bytes, stream, out, &kg);
}

int ltdi_orbits_init_tables(const ltdi_orbit_desc *desc, const double *d_R, const double *d_L, void *d_tables,
                            size_t bytes, void *stream, ltdi_orbits **out)
{
    if (!desc || desc->mode != LTDI_ORBIT_TABLES || !d_R || !d_L) return LTDI_EINVAL;
    return orbits_common(desc, d_R, d_L, d_tables, bytes, stream, out);
}

int ltdi_orbits_prepare_bytes(const ltdi_orbit_desc *desc, int lagrange_order, size_t *bytes)
{
    if (!desc_ok(desc) || !order_ok(lagrange_order) || !bytes) return LTDI_EINVAL;
    if (!fast_order(lagrange_order)) { *bytes = 0; return LTDI_OK; }
    const int64_t tiles = (desc->n + FAST_TCA - 1) / FAST_TCA;
    *bytes = ((size_t)tiles * FAST_NA * (FAST_ANC_DOUBLES(lagrange_order + 1) + 4 + (lagrange_order + 1)) * sizeof(double) + 255) / 256 * 256;
    return LTDI_OK;
}

int ltdi_orbits_prepare(ltdi_orbits *orb, int gen, int lagrange_order, void *d_buf, size_t bytes, void *stream)
{
    if (!orb || !gen_ok(gen) || !order_ok(lagrange_order)) return LTDI_EINVAL;
    if (!fast_order(lagrange_order)) return LTDI_OK;   /* the other orders build their weights per sample */
    size_t need = 0;
    ltdi_orbits_prepare_bytes(&orb->desc, lagrange_order, &need);
    if (!d_buf || (uintptr_t)d_buf % 16) return LTDI_EINVAL;
    if (bytes < need) return LTDI_EWORKSPACE;
    DeviceState *ds = nullptr;
    int rc = device_state(&ds);
    if (rc) return rc;
    const ltdi_orbit_desc &d = orb->desc;
    const int M = lagrange_order + 1;
    const Margins m15 = compute_margins(d, LTDI_GEN_15, lagrange_order, 0), m20 = compute_margins(d, LTDI_GEN_20, lagrange_order, 0);
    if (m20.m2 > 4096 || m20.m1 > 8192) return LTDI_OK; /* shapes the tuned kernels do not cover */
    FastParams p;
    std::memset(&p, 0, sizeof p);
    p.tab = orb->d_tab; p.stride = orb->stride; p.n = d.n; p.t0 = d.t0; p.dt = d.dt; p.inv_dt = 1.0 / d.dt;
    p.gen = gen; p.m1 = m20.m1; p.m2 = m20.m2; p.m2_15 = m15.m2; p.m2_20 = m20.m2;
    const int64_t tiles = (d.n + FAST_TCA - 1) / FAST_TCA;
    double *anc = (double *)d_buf, *hdr = anc + (size_t)tiles * FAST_NA * FAST_ANC_DOUBLES(M);
    /* w'' for the orbit objects whose responses run on the second-order instances (caller's tables, numerical orbit files);
     * a nested call on an analytic orbit builds its own anchors */
    const bool has2 = d.mode == LTDI_ORBIT_TABLES || d.mode == LTDI_ORBIT_KNOTS;
    double *anc2 = has2 ? hdr + (size_t)tiles * FAST_NA * 4 : nullptr;
    {
        ProfScope ps(LTDI_KERNEL_ANCHOR, (cudaStream_t)stream);
        if (M == 32) anchor_kernel<32><<<(unsigned)tiles, 64, 0, (cudaStream_t)stream>>>(p, anc, hdr, anc2);
        else anchor_kernel<10><<<(unsigned)tiles, 64, 0, (cudaStream_t)stream>>>(p, anc, hdr, anc2);
    }
    orb->anc_has2 = has2;
    count_launch();
    LTDI_CUDA_OK(cudaGetLastError());
    orb->d_anc = anc;
    orb->anc_gen = gen;
    orb->anc_M = M;
    return LTDI_OK;
}

int ltdi_orbits_destroy(ltdi_orbits *orb)
{
    delete orb;
    return LTDI_OK;
}

int64_t ltdi_orbits_stride(const ltdi_orbits *orb) { return orb ? orb->stride : 0; }
const double *ltdi_orbits_tables(const ltdi_orbits *orb) { return orb ? orb->d_tab : nullptr; }

int ltdi_margins(const ltdi_orbit_desc *desc, int gen, int lagrange_order, int fd_order, int64_t *lo, int64_t *hi)
{
    if (!desc_ok(desc) || !gen_ok(gen) || !order_ok(lagrange_order) || !lo || !hi) return LTDI_EINVAL;
    if (fd_order != 0 && fd_order != 2 && fd_order != 4) return LTDI_EINVAL;
    const Margins m = compute_margins(*desc, gen, lagrange_order, fd_order);
    *lo = m.lo;
    *hi = m.hi;
    return LTDI_OK;
}

int ltdi_link_margins(const ltdi_orbit_desc *desc, int lagrange_order, int fd_order, int64_t *lo, int64_t *hi)
{
    if (!desc_ok(desc) || !order_ok(lagrange_order) || !lo || !hi) return LTDI_EINVAL;
    if (fd_order != 0 && fd_order != 2 && fd_order != 4) return LTDI_EINVAL;
    const Margins m = compute_margins(*desc, LTDI_GEN_15, lagrange_order, fd_order);
    *lo = m.m1 + m.w;
    *hi = m.m1 + m.w;
    return LTDI_OK;
}

int ltdi_hyb_time(double f_hyb_hz, double mchirp_s, double t_c, double *t_hyb)
{
    if (!t_hyb || !(f_hyb_hz > 0.0) || !(mchirp_s > 0.0)) return LTDI_EINVAL;
    *t_hyb = t_c - 5.0 * std::pow(8.0 * 3.14159265358979323846 * f_hyb_hz, -8.0 / 3.0) * std::pow(mchirp_s, -5.0 / 3.0);
    return LTDI_OK;
}

int ltdi_workspace_bytes(int which, int64_t n, int64_t batch, int gen, int lagrange_order, size_t *bytes)
{
    if (which < LTDI_RESPONSE_FULL || which > LTDI_RESPONSE_HYBRID || n < 1 || batch < 1 || !bytes) return LTDI_EINVAL;
    if (!gen_ok(gen) || !order_ok(lagrange_order)) return LTDI_EINVAL;
    const size_t dbl = fast_order(lagrange_order) ? fast_layout(which, n, batch, lagrange_order + 1).total : work_doubles(batch);
    *bytes = (dbl * sizeof(double) + 255) / 256 * 256;
    return LTDI_OK;
}

int ltdi_response_full(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                       const ltdi_source *h_src, int gen, int lagrange_order, double *d_A, double *d_E, double *d_T,
                       double *d_XYZ, double *d_y, void *d_work, size_t work_bytes, void *stream)
{
    return run_response(LTDI_RESPONSE_FULL, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, 0, nullptr, 0,
                        d_A, d_E, d_T, d_XYZ, d_y, d_work, work_bytes, stream);
}

int ltdi_response_full_nested(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                              const ltdi_source *h_src, int gen, int lagrange_order, int nested_order, double *d_A,
                              double *d_E, double *d_T, double *d_XYZ, double *d_y, void *d_work, size_t work_bytes,
                              void *stream)
{
    if (nested_order == 0) return LTDI_EINVAL;
    return run_response(LTDI_RESPONSE_FULL, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, 0, nullptr, 0,
                        d_A, d_E, d_T, d_XYZ, d_y, d_work, work_bytes, stream, 1, LTDI_LFA_CENTRAL, nested_order);
}

int ltdi_response_full_chirp(const ltdi_orbits *orb, const ltdi_chirp *h_wav, int64_t ld, int64_t batch,
                             const ltdi_source *h_src, int gen, int lagrange_order, double *d_A, double *d_E, double *d_T,
                             double *d_XYZ, double *d_y, void *d_work, size_t work_bytes, void *stream)
{
    if (!h_wav) return LTDI_EINVAL;
    return run_response(LTDI_RESPONSE_FULL, orb, nullptr, nullptr, ld, batch, h_src, gen, lagrange_order, 0, nullptr, 0,
                        d_A, d_E, d_T, d_XYZ, d_y, d_work, work_bytes, stream, 1, LTDI_LFA_CENTRAL, 0, h_wav);
}

int ltdi_waveform_chirp(const ltdi_chirp *h_wav, int64_t batch, double t0, double dt, int64_t n, int64_t ld, double *d_hp,
                        double *d_hc, void *d_work, size_t work_bytes, void *stream)
{
    if (!h_wav || !d_hp || !d_hc || !d_work || batch < 1 || batch > 65535 || n < 1 || ld < n || !(dt > 0.0)) return LTDI_EINVAL;
    if (work_bytes < (size_t)batch * sizeof(ChirpDev)) return LTDI_EWORKSPACE;
    if ((uintptr_t)d_work % 16) return LTDI_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int rc = upload_chirps(h_wav, batch, t0, (ChirpDev *)d_work, st);
    if (rc) return rc;
    chirp_grid_kernel<<<dim3((unsigned)((n + 255) / 256), (unsigned)batch), 256, 0, st>>>((const ChirpDev *)d_work, dt, n, ld, d_hp, d_hc);
    count_launch();
    LTDI_CUDA_OK(cudaGetLastError());
    return LTDI_OK;
}

int ltdi_waveform_ecc(const double *d_tab, int64_t nk, const double *h_par, int nharm, int64_t batch, double t0, double dt,
                      int64_t n, int64_t ld, double *d_hp, double *d_hc, void *d_work, size_t work_bytes, void *stream)
{
    if (!d_tab || !h_par || !d_hp || !d_hc || !d_work || nk < 2 || nharm < 1 || nharm > 64 || batch < 1 || batch > 65535 ||
        n < 1 || ld < n || !(dt > 0.0))
        return LTDI_EINVAL;
    if (work_bytes < (size_t)batch * sizeof(EccDev)) return LTDI_EWORKSPACE;
    if ((uintptr_t)d_work % 16) return LTDI_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    EccDev *d_wav = (EccDev *)d_work;
    EccArgs *a = new (std::nothrow) EccArgs;
    if (!a) return LTDI_EINVAL;
    for (int64_t b0 = 0; b0 < batch; b0 += LTDI_ECC_SLICE) {
        const int cnt = (int)std::min<int64_t>(LTDI_ECC_SLICE, batch - b0);
        for (int i = 0; i < cnt; ++i)
            if (ecc_fill(h_par + 6 * (b0 + i), &a->v[i])) { delete a; return LTDI_EINVAL; }
        unpack_ecc_kernel<<<(cnt * LTDI_ECC_STRIDE + 127) / 128, 128, 0, st>>>(*a, cnt, d_wav + b0);
        count_launch();
        if (cudaGetLastError() != cudaSuccess) { delete a; return LTDI_ECUDA; }
    }
    delete a;
    ecc_grid_kernel<<<dim3((unsigned)((n + 127) / 128), (unsigned)batch), 128, 0, st>>>(d_tab, nk, d_wav, nharm, t0, dt, n, ld, d_hp, d_hc);
    count_launch();
    LTDI_CUDA_OK(cudaGetLastError());
    return LTDI_OK;
}

int ltdi_response_lfa(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                      const ltdi_source *h_src, int gen, int lagrange_order, int fd_order, double *d_A, double *d_E,
                      double *d_T, double *d_XYZ, double *d_y, void *d_work, size_t work_bytes, void *stream)
{
    return run_response(LTDI_RESPONSE_LFA, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, fd_order, nullptr,
                        0, d_A, d_E, d_T, d_XYZ, d_y, d_work, work_bytes, stream);
}

int ltdi_response_lfa_ext(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                          const ltdi_source *h_src, int gen, int lagrange_order, int fd_order, int terms, int point,
                          double *d_A, double *d_E, double *d_T, double *d_XYZ, double *d_y, void *d_work,
                          size_t work_bytes, void *stream)
{
    return run_response(LTDI_RESPONSE_LFA, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, fd_order, nullptr,
                        0, d_A, d_E, d_T, d_XYZ, d_y, d_work, work_bytes, stream, terms, point);
}

int ltdi_response_lfa6(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                       const ltdi_source *h_src, int gen, int lagrange_order, int fd_order, double *d_A, double *d_E,
                       double *d_T, double *d_XYZ, double *d_y, void *d_work, size_t work_bytes, void *stream)
{
    return run_response(LTDI_RESPONSE_LFA, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, fd_order, nullptr,
                        0, d_A, d_E, d_T, d_XYZ, d_y, d_work, work_bytes, stream, 1, LTDI_LFA_CENTRAL, 0, nullptr, 1);
}

int ltdi_response_full_sagnac(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                              const ltdi_source *h_src, int gen, int lagrange_order, double *d_A, double *d_E, double *d_T,
                              double *d_abc, double *d_y, void *d_work, size_t work_bytes, void *stream)
{
    return run_response(LTDI_RESPONSE_FULL, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, 0, nullptr, 0, d_A,
                        d_E, d_T, d_abc, d_y, d_work, work_bytes, stream, 1, LTDI_LFA_CENTRAL, 0, nullptr, 0, 1);
}

int ltdi_margins_lfa6(const ltdi_orbit_desc *desc, int gen, int lagrange_order, int fd_order, int64_t *lo, int64_t *hi)
{
    if (fd_order != 2 && fd_order != 4) return LTDI_EINVAL;
    const int rc = ltdi_margins(desc, gen, lagrange_order, fd_order, lo, hi);
    if (rc) return rc;
    if (gen == LTDI_GEN_20) { *lo += 1; *hi += 1; }
    return LTDI_OK;
}

int ltdi_margins_lfa_ext(const ltdi_orbit_desc *desc, int gen, int lagrange_order, int fd_order, int terms, int64_t *lo,
                         int64_t *hi)
{
    if (terms < 1 || terms > 2 || (fd_order != 2 && fd_order != 4)) return LTDI_EINVAL;
    const int rc = ltdi_margins(desc, gen, lagrange_order, fd_order, lo, hi);
    if (rc) return rc;
    *lo += terms - 1;
    *hi += terms - 1;
    return LTDI_OK;
}

int ltdi_response_hybrid(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                         const ltdi_source *h_src, int gen, int lagrange_order, int fd_order,
                         const ltdi_hybrid *h_hyb, int64_t n_hyb, double *d_A, double *d_E, double *d_T,
                         double *d_XYZ, double *d_y, void *d_work, size_t work_bytes, void *stream)
{
    return run_response(LTDI_RESPONSE_HYBRID, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, fd_order,
                        h_hyb, n_hyb, d_A, d_E, d_T, d_XYZ, d_y, d_work, work_bytes, stream);
}

int64_t ltdi_launch_count(void) { return g_launches.load(); }

int ltdi_profile_enable(int on)
{
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_prof_on = on != 0;
    return LTDI_OK;
}

int ltdi_profile_read(int kernel, int which, double *total_ms, int64_t *launches)
{
    if (kernel < 0 || kernel >= LTDI_KERNEL_COUNT || which < 0 || which > 2 || !total_ms || !launches) return LTDI_EINVAL;
    std::lock_guard<std::mutex> lk(g_prof_mu);
    for (const ProfPair &pr : g_prof_pending) {
        float ms = 0.f;
        if (cudaEventSynchronize(pr.e1) != cudaSuccess || cudaEventElapsedTime(&ms, pr.e0, pr.e1) != cudaSuccess) {
            (void)cudaGetLastError();
            return LTDI_ECUDA;
        }
        g_prof_ms[pr.id] += ms;
        g_prof_n[pr.id] += 1;
        g_prof_pool.push_back(pr.e0);
        g_prof_pool.push_back(pr.e1);
    }
    g_prof_pending.clear();
    *total_ms = g_prof_ms[kernel + LTDI_KERNEL_COUNT * which];
    *launches = g_prof_n[kernel + LTDI_KERNEL_COUNT * which];
    return LTDI_OK;
}

int ltdi_profile_reset(void)
{
    double ms; int64_t n;
    const int rc = ltdi_profile_read(0, 0, &ms, &n);   /* drains pending pairs */
    std::lock_guard<std::mutex> lk(g_prof_mu);
    for (int i = 0; i < 3 * LTDI_KERNEL_COUNT; ++i) { g_prof_ms[i] = 0.0; g_prof_n[i] = 0; }
    return rc;
}
int ltdi_profile_slow_tiles(int64_t *count, int reset)
{
    if (!count) return LTDI_EINVAL;
    unsigned long long v = 0;
    LTDI_CUDA_OK(cudaMemcpyFromSymbol(&v, d_slow_tiles, sizeof v));
    *count = (int64_t)v;
    if (reset) {
        v = 0;
        LTDI_CUDA_OK(cudaMemcpyToSymbol(d_slow_tiles, &v, sizeof v));
    }
    return LTDI_OK;
}
const char *ltdi_version(void) { return "lisatdi-b200 0.1 (sm_100a, fp64)"; }

} // extern "C"

// ---- ltdi_response_static: the responses with the scratch in a file-scope device array (no allocation anywhere) --------
// In host code `g_static_scratch` is a host-side stand-in for the symbol, not a device address: the address the kernels
// get comes from cudaGetSymbolAddress, looked up once per device with that device current.
static __device__ __align__(256) double g_static_scratch[LTDI_STATIC_SCRATCH_BYTES / sizeof(double)];
static std::mutex g_static_mu;
static void *g_static_ptr[64];   /* device address of g_static_scratch on device i, or nullptr before its set-up */

static int static_scratch(void **out)
{
    int dev = 0;
    LTDI_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return LTDI_EUNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        DeviceState *ds = nullptr;   /* the library's one-time set-up of the device (constant tables, side stream) */
        const int rc = device_state(&ds);
        if (rc) return rc;
        void *p = nullptr;
        LTDI_CUDA_OK(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (uintptr_t)p % 256) return LTDI_ECUDA;
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return LTDI_OK;
}

extern "C" int ltdi_response_static(int which, const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                                    int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, int fd_order,
                                    const ltdi_hybrid *h_hyb, int64_t n_hyb, double *d_A, double *d_E, double *d_T,
                                    void *stream)
{
    if (which < LTDI_RESPONSE_FULL || which > LTDI_RESPONSE_HYBRID || !orb || batch < 1) return LTDI_EINVAL;
    size_t need = 0;
    const int rc = ltdi_workspace_bytes(which, orb->desc.n, batch, gen, lagrange_order, &need);
    if (rc) return rc;
    if (need > LTDI_STATIC_SCRATCH_BYTES) {
        if (getenv("LTDI_DEBUG"))
            fprintf(stderr, "lisatdi: ltdi_response_static needs %zu bytes of scratch, the static array holds %zu\n", need,
                    (size_t)LTDI_STATIC_SCRATCH_BYTES);
        return LTDI_EWORKSPACE;
    }
    void *d_work = nullptr;
    const int src = static_scratch(&d_work);
    if (src) return src;
    return run_response(which, orb, d_hp, d_hc, ld, batch, h_src, gen, lagrange_order, fd_order, h_hyb, n_hyb, d_A, d_E, d_T,
                        nullptr, nullptr, d_work, LTDI_STATIC_SCRATCH_BYTES, stream);
}
