// rc_api.cu — the C ABI of include/rc.h: context, validation, workspace layout, launch sequence.
// Host logic only; every arithmetic step of the path runs in rc_kernels.cu.  No CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/rc.h"
#include "rc_internal.h"

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

// Launch knobs (rc_set_tuning): measurement and test aids; none changes a result beyond rounding unless noted.
struct Tuning {
    int variant = -1;      // march_variant 0..4: register-ring depth / occupancy of the march; -1: chosen per cascade
    int patch_log2 = -1;   // 2..5: lane patch width 2^n for cascades >= patch_from; -1: chosen per cascade (choose_patch)
    int patch_from = 0;
    int cpw_from = 3;      // cascades >= this run one child direction per warp; -1: off
    bool cpw_forced = false;
    float tau_cut = 126.f; // early-exit threshold on tau log2(e); 126: the fp32 transmittance is exactly 0 (below: changes J)
    int bands = 0;         // L2 banding: number of bands; 0: from the L2 budget
    double l2_mb = 72.0;   // L2 budget of one wavelength batch of packed chi, S
    int sparse = -1;       // distance-field march: -1 automatic (> 2/3 of the cells empty), 0 never, 1 whenever analysed
    int graph = 1;         // CUDA graph replay on small grids
    int sparse_mode = 1;   // fan march variant, 0..3 (blocks of 8 / 4 / 2 warps, or 4 warps at 128 registers)
    int list_b = 0;        // wavelength batches per warp of the march over hit lists: 0 from the L2 footprint, or 1, 2, 4, 8
    int pipeline = 1;      // rc_solve_J_host: two halves of the wavelength batches, copies overlapped with the other half's solve
    int lists = 1;         // hit lists for the sparse march when the caller lends a buffer (rc_set_sparse_workspace): 0 never
    int sorted = -1;       // lanes from sorted quads: -1 where the geometry says it pays, 0 never, 1 wherever possible
};

struct CascadePlan {
    bool fix = false;           // bilinear fix: 16 tables per direction, lanes = one parity class, packed with spacing 2s
    size_t subdir_off = 0;      // fix: unit directions of the sub-rays [ndir*16] float2
    bool banded = false;        // marched band by band (Plan::nbands launches per direction half)
    int pw_log2 = 5;            // lane patch of the march: 2^pw_log2 probes wide, 32 >> pw_log2 high
    double patch_util = 1.0;    // estimated lock-step lane utilisation of that patch shape
    bool sorted = false;        // lanes = 8 quads of probes taken from a list sorted by ray length (per block of 8 direction groups)
    int qpad = 0;               // entries per block of direction groups (quads, padded to a multiple of 8)
    size_t qlist_off = 0;       // [ngroups / 8][qpad] uint16
    long long ndir = 0;         // 4^(i+1)
    bool empty = true;          // interval starts beyond the box diagonal: no ray of it is inside
    long long slots = 0;        // step-table capacity, all directions
    size_t off_off = 0, cnt_off = 0, steps_off = 0, xy_off = 0;  // byte offsets into the workspace
    double ta = 0, tb = 0;
};

struct Plan {
    int nx = 0, ny = 0, L = 0, ncasc = 0;
    int LV = 1, nb = 1, Lpad = 1;   // wavelengths per lane, batches, nb * LV
    int NM = 1;                     // inclinations (2.5D); a lane carries LV * NM channels
    int nbands = 1, band_axis = 0;  // L2 banding of the long-ray cascades (1 = off); axis 0 = rows, 1 = columns
    size_t state = 0;               // parked ray state of the banded launches
    bool line = false;              // velocity-dependent line mode: chiT holds 6 packed line parameters per cell
    size_t xls = 0;                 // line mode: scaled wavelengths [Lpad]
    // sparsity: flagged probes per cascade (bytes), compacted patch lists, and the distance field
    size_t pflag[RC_MAX_CASCADES] = {0}, plist[RC_MAX_CASCADES] = {0}, pmark = 0, pcount = 0;
    int plist_cap[RC_MAX_CASCADES] = {0};
    size_t occ8 = 0, d1 = 0, dist = 0;
    CascadePlan c[RC_MAX_CASCADES];
    bool multi_pack = false;        // small grids: per-cascade packed arrays, one pack launch per solve
    size_t chiT_c[RC_MAX_CASCADES] = {0}, ST_c[RC_MAX_CASCADES] = {0};
    size_t chiT = 0, ST = 0, A[2] = {0, 0}, Jpart = 0, bc_below = 0, bc_above = 0, weights = 0, flag = 0;
    size_t io_chi = 0, io_eta = 0, io_J = 0;
    size_t total = 0;
};

}  // namespace

struct rc_ctx {
    rc_config cfg{};
    cudaStream_t stream = nullptr;
    char *ws = nullptr;
    size_t ws_bytes = 0;
    const float *chi = nullptr, *eta = nullptr;
    const float *line = nullptr;  // line mode: [ny][nx][6], borrowed
    Plan plan{};
    bool have_atm = false;
    int tab_nx = 0, tab_ny = 0;  // shape the step tables in the workspace were built for
    bool host_io = false;
    // CUDA graph of the launch sequence of small grids (rc_solve_J) and what it was captured for
    struct GraphKey { const void *J, *chi, *eta, *line, *ws; int nx, ny, L, nm, sparse, tune_gen; size_t total; float f[8], w[8]; };
    GraphKey graph_key{};
    cudaGraphExec_t graph_exec = nullptr;
    int tune_gen = 0;  // counts rc_set_tuning calls: a knob may change launch variants and workspace offsets
    cudaStream_t cap_stream = nullptr;
    cudaStream_t copy_stream = nullptr;   // rc_solve_J_host's pipeline: the other half's copies
    cudaEvent_t pipe_ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    // sparsity
    bool active_set = false;   // rc_set_active_cells: flagged probes per cascade are in the workspace
    bool lists_dirty = false;  // the compacted patch lists must be rebuilt (before the next solve; synchronises once)
    int npatch_act[RC_MAX_CASCADES] = {0};
    int list_version = 0;
    bool sparse = false;       // rc_analyse_atmosphere found the atmosphere mostly empty: the march walks the distance field
    // hit lists of the sparse march (valid while `sparse`): in the caller's second buffer (rc_set_sparse_workspace)
    char *sws = nullptr;
    size_t sws_bytes = 0;
    bool lists = false;
    int64_t list_bytes = 0;
    bool lists_built = false;  // the buffer holds lists for the occupancy map stored at its start: an analysis that finds the same map keeps them
    int list_b = 1;            // wavelength batches per warp of the march over hit lists
    size_t hit_off[RC_MAX_CASCADES] = {0}, hit_list[RC_MAX_CASCADES] = {0};  // byte offsets into sws
    bool count_walked = false; // the solve being enqueued counts the segments it integrates (rc_count_walked)
    bool analysed = false;     // rc_analyse_atmosphere has been used on this context (rc_solve_J_host then repeats it)
    std::vector<float> xl_stage;  // line mode: host copy of the scaled wavelengths (kept alive for the async upload)
    bool xl_on_device = false;    // the workspace holds xl_stage at plan.xls: false after anything that moves or overwrites that region
                                  // (another workspace, a new plan, a GivenFs atmosphere whose packed arrays share the bytes)
    Tuning tune{};
    // 2.5D inclination quadrature (rc_set_inclinations); nm = 1, f = w = 1: flatland
    int nm = 1;
    float incl_f[8] = {1, 1, 1, 1, 1, 1, 1, 1}, incl_w[8] = {1, 0, 0, 0, 0, 0, 0, 0};
    std::vector<std::vector<long long>> off_host;  // kept alive for the async uploads
    std::vector<std::vector<unsigned short>> qlist_host;
    std::vector<float> stage;                      // host staging for boundary / weights
    // timing: `nsets` rings of (2 per cascade + 2) events; solve number n records into set n % nsets
    int nsets = 0;
    long long solves_timed = 0;
    std::vector<cudaEvent_t> ev;
    rc_stats stats{};
    char err[512] = {0};
};

namespace {

int fail(rc_ctx *ctx, int code, const char *fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define RC_CUDA(ctx, call)                                                                       \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess)                                                                   \
            return fail(ctx, RC_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                                     \
    } while (0)

// Interval ends, PAPER.md:171-176 (eq. 12-13) with alpha = 2: t_i = c0 (4^i - 1)/3.
double t_of(int i, double c0) { return c0 * (std::pow(4.0, (double)i) - 1.0) / 3.0; }

bool shape_ok(const rc_config &cfg, int nx, int ny, int L) {
    if (nx <= 0 || ny <= 0 || L <= 0 || nx > RC_MAX_DIM || ny > RC_MAX_DIM) return false;
    const int m = 1 << (cfg.ncascades - 1);
    return nx % m == 0 && ny % m == 0;
}

// Shape of the 32-probe patch one warp marches in lock step.  All lanes walk until the patch's last
// ray has left the box, so the patch should hold probes whose rays have similar in-box lengths:
// estimated here from the geometry alone (ray length to the box edge, clipped to the interval) for
// the candidate shapes 32x1 .. 4x8, over a sample of directions.  Wider patches gather longer
// contiguous runs, so the widest shape within 2 % of the best utilisation wins.
int choose_patch(int nx, int ny, int i, double ta, double tb, double *util, int step = 1) {  // step 2: one parity class (bilinear fix)
    *util = 1.0;
    const int s = 1 << i, npx = (nx >> i) / step, npy = (ny >> i) / step;
    int widest = 5;
    while (widest > 0 && (1 << widest) > npx) widest--;
    if (std::fmin(tb, std::hypot((double)nx, (double)ny)) <= std::min(nx, ny) / 16.0) return widest;
    const long long ndir = 1LL << (2 * (i + 1));
    const int nsample = (int)std::min<long long>(ndir, 32);
    std::vector<double> len((size_t)npx * npy);
    double total = 0.0, cost[6] = {0, 0, 0, 0, 0, 0};
    const int narrowest = std::min(widest, 2);
    for (int n = 0; n < nsample; n++) {
        const long long k = (2 * n + 1) * ndir / (2 * nsample);
        const double th = 2.0 * M_PI * ((double)k + 0.5) / (double)ndir, cx = std::cos(th), sy = std::sin(th);
        for (int b = 0; b < npy; b++)
            for (int a = 0; a < npx; a++) {
                const double X = (step * a + 0.5) * s, Y = (step * b + 0.5) * s;
                const double te = std::fmin(cx > 0 ? (nx - X) / cx : -X / cx, sy > 0 ? (ny - Y) / sy : -Y / sy);
                const double l = std::fmax(std::fmin(te, tb) - ta, 0.0) * (std::fabs(cx) + std::fabs(sy));
                len[(size_t)b * npx + a] = l;
                total += l;
            }
        for (int c = narrowest; c <= widest; c++) {
            const int pw = 1 << c, ph = 32 >> c;
            for (int b0 = 0; b0 < npy; b0 += ph)
                for (int a0 = 0; a0 < npx; a0 += pw) {
                    double m = 0.0;
                    for (int b = b0; b < std::min(b0 + ph, npy); b++)
                        for (int a = a0; a < std::min(a0 + pw, npx); a++) m = std::fmax(m, len[(size_t)b * npx + a]);
                    cost[c] += 32.0 * m;
                }
        }
    }
    if (!(total > 0.0)) return widest;
    double best = 0.0;
    for (int c = narrowest; c <= widest; c++) best = std::fmax(best, total / cost[c]);
    for (int c = widest; c >= narrowest; c--)
        if (total / cost[c] >= best - 0.02) { *util = total / cost[c]; return c; }
    return widest;
}

// Sorted quads: the lanes of a warp need not be a rectangle of probes - the gathers only want runs of 4 x-adjacent
// probes (one 128-byte line at 8 wavelengths per lane).  For a block of 8 direction groups (32 adjacent directions) the
// quads of the lattice are ordered by the length of their longest ray inside the box (geometry alone, as in
// choose_patch) and a warp takes 8 consecutive quads: its 32 lock-step lanes then finish almost together wherever the
// quads sit.  Returns the estimated utilisation; fills `list` ([nblocks][qpad], 0xffff = padding) when given.
// `step` = 2: the lattice of one parity class of the bilinear fix (every other probe per axis).
double sorted_quads(int nx, int ny, int i, double ta, double tb, int qpad, std::vector<unsigned short> *list, int step = 1) {
    const int s = 1 << i, npx = (nx >> i) / step, npy = (ny >> i) / step, qx = npx / 4, nq = qx * npy;
    const long long ndir = 1LL << (2 * (i + 1));
    const int nblocks = (int)(ndir / 32);
    if (list) list->assign((size_t)nblocks * qpad, (unsigned short)0xffff);
    const int stride = list ? 1 : std::max(1, nblocks / 32);  // the estimate looks at a sample of the blocks
    std::vector<double> key((size_t)nq);
    std::vector<int> order((size_t)nq);
    double total = 0.0, cost = 0.0;
    for (int blk = 0; blk < nblocks; blk += stride) {
        const double th = 2.0 * M_PI * (32.0 * blk + 16.0) / (double)ndir, cx = std::cos(th), sy = std::sin(th);
        for (int b = 0; b < npy; b++)
            for (int q = 0; q < qx; q++) {
                double m = 0.0;
                for (int j = 0; j < 4; j++) {
                    const double X = (step * (4 * q + j) + 0.5) * s, Y = (step * b + 0.5) * s;
                    const double te = std::fmin(cx > 0 ? (nx - X) / cx : -X / cx, sy > 0 ? (ny - Y) / sy : -Y / sy);
                    const double l = std::fmax(std::fmin(te, tb) - ta, 0.0) * (std::fabs(cx) + std::fabs(sy));
                    total += l;
                    m = std::fmax(m, l);
                }
                key[(size_t)b * qx + q] = m;
            }
        for (int q = 0; q < nq; q++) order[q] = q;
        std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return key[x] > key[y]; });
        for (int q0 = 0; q0 < nq; q0 += 8) cost += 32.0 * key[order[q0]];
        if (list)
            for (int q = 0; q < nq; q++) (*list)[(size_t)blk * qpad + q] = (unsigned short)order[q];
    }
    return cost > 0.0 ? total / cost : 1.0;
}

// Wavelengths per lane: a lane carries LV * nm <= 8 channels (registers).
int choose_lv(const rc_config &cfg, int L, int nm) {
    const int cap = 8 / nm;
    if ((cfg.lambda_batch == 1 || cfg.lambda_batch == 2 || cfg.lambda_batch == 4 || cfg.lambda_batch == 8) &&
        cfg.lambda_batch <= cap)
        return cfg.lambda_batch;
    int lv = 1;
    while (lv < L && lv < cap) lv <<= 1;
    return lv;
}

// Workspace layout for a shape.  When `offs` is given, also fills the per-direction slot offsets.
bool make_plan_uncached(const rc_config &cfg, const Tuning &tune, int nm, bool line, int nx, int ny, int L, bool host_io, Plan &P,
                        std::vector<std::vector<long long>> *offs) {
    if (!shape_ok(cfg, nx, ny, L)) return false;
    P = Plan{};
    P.nx = nx; P.ny = ny; P.L = L; P.ncasc = cfg.ncascades;
    P.NM = nm;
    P.line = line;
    P.LV = choose_lv(cfg, L, nm);
    P.nb = (L + P.LV - 1) / P.LV;
    P.Lpad = P.nb * P.LV;
    const size_t ncell = (size_t)nx * ny;
    const double diag = std::sqrt((double)nx * nx + (double)ny * ny);
    const int top = cfg.ncascades - 1;
    size_t cur = 0;
    if (offs) offs->assign(cfg.ncascades, {});
    for (int i = 0; i <= top; i++) {
        CascadePlan &c = P.c[i];
        c.ndir = 1LL << (2 * (i + 1));
        c.ta = t_of(i, cfg.c0_interval);
        c.tb = i == top ? INFINITY : t_of(i + 1, cfg.c0_interval);
        c.empty = !(c.ta < diag);
        c.slots = 0;
        c.pw_log2 = 5;
        while (c.pw_log2 > 0 && (1 << c.pw_log2) > (nx >> i)) c.pw_log2--;
        if (c.empty) continue;
        c.fix = (cfg.flags & RC_BILINEAR_FIX) != 0 && i < top;
        c.pw_log2 = choose_patch(nx, ny, i, c.ta, c.tb, &c.patch_util, c.fix && (nx >> i) >= 2 && (ny >> i) >= 2 ? 2 : 1);
        std::vector<long long> local;
        std::vector<long long> &o = offs ? (*offs)[i] : local;
        const int nsub = c.fix ? 16 : 1;
        o.resize((size_t)c.ndir * nsub + 1);
        long long acc = 0;
        for (long long k = 0; k < c.ndir * nsub; k++) {
            o[(size_t)k] = acc;
            long long n;
            if (c.fix) {
                // sub-ray from p + t_i w to q + t_(i+1) w: at most (t_(i+1) - t_i) + 1.5 sqrt2 s long, clipped by the box
                const double len = std::fmin(c.tb - c.ta + 2.2 * (1 << i), diag + 2.0 * (1 << i));
                n = (long long)(len * 1.4143) + 8;
            } else if (i == 0) {
                const double cells = std::isinf(c.tb) ? (double)std::min(nx, ny)
                                                      : std::min((double)std::min(nx, ny), std::ceil(c.tb / std::sqrt(2.0) + 0.5) + 1.0);
                n = (long long)cells;
            } else {
                const double th = 2.0 * M_PI * ((double)k + 0.5) / (double)c.ndir;  // (nsub == 1 here)
                const double wx = std::fabs(std::cos(th)), wy = std::fabs(std::sin(th));
                const double tb = std::fmin(c.tb, std::fmin(nx / wx, ny / wy));
                n = tb > c.ta ? (long long)((tb - c.ta) * (wx + wy)) + 6 : 0;
            }
            acc += n;
        }
        o[(size_t)c.ndir * nsub] = acc;
        c.slots = acc;
        c.off_off = cur;   cur = align_up(cur + sizeof(long long) * ((size_t)c.ndir * nsub + 1));
        c.cnt_off = cur;   cur = align_up(cur + sizeof(int) * (size_t)c.ndir * nsub);
        if (c.fix) { c.subdir_off = cur; cur = align_up(cur + sizeof(float2) * (size_t)c.ndir * 16); }
        // + 16 entries: the march loop reads the table up to 2 x (ring depth) entries past the last step
        c.steps_off = cur; cur = align_up(cur + sizeof(rc::Step) * ((size_t)acc + 16));
        c.xy_off = cur;    cur = align_up(cur + sizeof(rc::StepXY) * ((size_t)acc + 16));
    }
    const size_t field = align_up(ncell * P.Lpad * sizeof(float));
    // L2 banding: one wavelength batch of packed chi and S is ncell * LV * 8 bytes; when that exceeds the
    // L2 budget the cascades with long rays are marched band by band
    {
        const double batch_mb = line ? 0.0 : (double)ncell * P.LV * 8.0 / (1 << 20);  // line mode: 24 B per cell
        P.nbands = (int)std::ceil(batch_mb / std::max(1.0, tune.l2_mb));
        if (tune.bands > 0) P.nbands = tune.bands;
        P.band_axis = nx > ny ? 1 : 0;
        const int n_axis = P.band_axis ? nx : ny;
        P.nbands = std::max(1, std::min(P.nbands, n_axis / 32));
        const int ext = (n_axis + P.nbands - 1) / P.nbands;
        bool any = false;
        for (int i = 1; i <= top; i++) {
            CascadePlan &c = P.c[i];
            // worth it for long rays only, and only while one warp's patch of probes is small against a
            // band (its lanes enter and leave a band at different steps: lock-step waste otherwise)
            const int patch_ext = (P.band_axis ? 1 << c.pw_log2 : 32 >> c.pw_log2) << i;
            // (long against the banded axis: the warps resident at one time stay within a fraction of a short ray's length of
            // one another, so short rays find their cells in L2 without bands - config 3, cascade 4: 80.5 ms banded, 63.9 not)
            const bool long_rays = std::fmin(c.tb, diag) - c.ta > 0.3 * n_axis;
            c.banded = P.nbands > 1 && !c.empty && !c.fix && ((long_rays && 4 * patch_ext <= ext) || (tune.bands > 0 && std::fmin(c.tb, diag) > 100.0));
            any = any || c.banded;
        }
        if (any) { P.state = cur; cur += 8 * field * P.NM; }
    }
    // lanes from sorted quads where that beats the best rectangular patch (long, clipped rays: the upper cascades)
    for (int i = 2; i <= top; i++) {
        CascadePlan &c = P.c[i];
        const int step = c.fix ? 2 : 1;   // bilinear fix: lanes are probes of one parity class
        const int npx = (nx >> i) / step, npy = (ny >> i) / step;
        const long long nq = (long long)(npx / 4) * npy;
        if (c.empty || c.banded || npx % 4 != 0 || nq < 8 || nq > 65535 || c.patch_util > 0.985 || tune.sorted == 0) continue;
        c.qpad = (int)((nq + 7) / 8 * 8);
        if (sorted_quads(nx, ny, i, c.ta, c.tb, c.qpad, nullptr, step) < c.patch_util + 0.015 && tune.sorted != 1) continue;
        c.sorted = true;
        c.qlist_off = cur; cur = align_up(cur + sizeof(unsigned short) * (size_t)(c.ndir / 32) * c.qpad);
    }
    {
        int cap_max = 1;
        for (int i = 0; i <= top; i++) {
            const size_t np = (size_t)(nx >> i) * (ny >> i);
            P.pflag[i] = cur; cur += align_up(np);
            // patches of 32 probes of any shape 2^k x 2^(5-k), x 4 parity classes with the bilinear fix
            P.plist_cap[i] = (int)std::min<size_t>(4 * (np / 32 + (size_t)(nx >> i) + (size_t)(ny >> i) + 4), 0x7fffffff);
            P.plist[i] = cur; cur += align_up(sizeof(int) * (size_t)P.plist_cap[i]);
            cap_max = std::max(cap_max, P.plist_cap[i]);
        }
        P.pmark = cur;  cur += align_up((size_t)cap_max);
        P.pcount = cur; cur += align_up(sizeof(int) * RC_MAX_CASCADES);
        P.occ8 = cur; cur += align_up(ncell);
        P.d1 = cur;   cur += align_up(ncell);
        P.dist = cur; cur += align_up(ncell);
    }
    if (line) {
        P.chiT = cur; cur += align_up(ncell * 6 * sizeof(float));
        P.xls = cur;  cur += align_up(2 * P.Lpad * sizeof(float));  // x_l sqrt(log2 e), then x_l
    } else {
        P.chiT = cur; cur += field;
        P.ST = cur;   cur += field;
        // launch-bound grids (config 0): every cascade gets its own packed arrays so that ONE launch packs for all of them
        static_assert(RC_MAX_CASCADES == 12, "PackParams::shifts");
        P.multi_pack = (long long)ncell * P.Lpad * P.NM <= (1LL << 21);
        for (int i = 0; i <= top && P.multi_pack; i++) {
            if (P.c[i].empty) continue;
            P.chiT_c[i] = cur; cur += field;
            P.ST_c[i] = cur;   cur += field;
        }
    }
    P.A[0] = cur; cur += field * P.NM;  // merged cascades hold every (wavelength, inclination) channel
    P.A[1] = cur; cur += field * P.NM;
    if (cfg.flags & RC_ACCUM_J) { P.Jpart = cur; cur += align_up(ncell * P.nb * sizeof(float)); }
    P.bc_below = cur; cur += align_up((size_t)P.Lpad * P.NM * sizeof(float));  // [Lpad][NM]: one value per channel
    P.bc_above = cur; cur += align_up((size_t)P.Lpad * P.NM * sizeof(float));
    P.weights = cur;  cur += align_up(P.Lpad * sizeof(float));
    P.flag = cur;     cur += 2 * ALIGN;  // scalar flags and counters (64-bit slots): [0..15] scratch, [16..31] segments walked per cascade, [32..43] flagged probes per cascade
    if (host_io) {
        const size_t io = align_up(ncell * L * sizeof(float));
        P.io_chi = cur; cur += io;
        P.io_eta = cur; cur += io;
        P.io_J = cur;   cur += (cfg.flags & RC_ACCUM_J) ? align_up(ncell * sizeof(float)) : io;
    }
    P.total = cur;
    return true;
}

// The plan is pure host arithmetic but not free (choose_patch); the last few are remembered.
bool make_plan(const rc_config &cfg, const Tuning &tune, int nm, bool line, int nx, int ny, int L, bool host_io, Plan &P,
               std::vector<std::vector<long long>> *offs) {
    struct Entry { double k[13]; Plan p; };
    static thread_local std::vector<Entry> cache;
    if (offs) return make_plan_uncached(cfg, tune, nm, line, nx, ny, L, host_io, P, offs);
    const double k[13] = {(double)cfg.ncascades, (double)cfg.lambda_batch, (double)cfg.flags, (double)nm, (double)line,
                          (double)nx, (double)ny, (double)L, (double)host_io, (double)cfg.c0_interval,
                          (double)tune.bands, tune.l2_mb, (double)tune.sorted};
    for (const Entry &e : cache)
        if (std::equal(k, k + 13, e.k)) { P = e.p; return true; }
    if (!make_plan_uncached(cfg, tune, nm, line, nx, ny, L, host_io, P, nullptr)) return false;
    if (cache.size() >= 16) cache.erase(cache.begin());
    Entry en;
    std::copy(k, k + 13, en.k);
    en.p = P;
    cache.push_back(en);
    return true;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Exported C ABI
// ------------------------------------------------------------------------------------------------
extern "C" {

const char *rc_version(void) { return "rc-b200 0.1 (sm_100a)"; }

const char *rc_last_error(const rc_ctx *ctx) { return ctx ? ctx->err : "null context"; }

int rc_plan_query(const rc_config *cfg, int ninclinations, int line_mode, int nx, int ny, int nlambda, rc_plan_info *out) {
    if (!cfg || !out) return RC_ERR_NULL_ARG;
    if (cfg->ncascades < 1 || cfg->ncascades > RC_MAX_CASCADES || !(cfg->c0_interval > 0.f) || !std::isfinite(cfg->c0_interval))
        return RC_ERR_BAD_VALUE;
    if (ninclinations != 1 && ninclinations != 2 && ninclinations != 4 && ninclinations != 8) return RC_ERR_BAD_VALUE;
    Plan P;
    if (!make_plan(*cfg, Tuning{}, ninclinations, line_mode != 0, nx, ny, nlambda, false, P, nullptr)) return RC_ERR_BAD_SHAPE;
    std::memset(out, 0, sizeof(*out));
    out->workspace_bytes = P.total;
    out->lambda_batch = P.LV;
    out->channels = P.LV * P.NM;
    out->nbatches = P.nb;
    out->nbands = P.nbands;
    out->band_axis = P.band_axis;
    for (int i = 0; i < cfg->ncascades; i++) {
        out->cascade_empty[i] = P.c[i].empty;
        out->cascade_banded[i] = P.c[i].banded;
        out->patch_w[i] = 1 << P.c[i].pw_log2;
        out->cascade_sorted[i] = P.c[i].sorted;
        out->lane_utilisation[i] = (float)(P.c[i].sorted ? sorted_quads(nx, ny, i, P.c[i].ta, P.c[i].tb, P.c[i].qpad, nullptr, P.c[i].fix ? 2 : 1) : P.c[i].patch_util);
        out->table_steps[i] = P.c[i].slots;
    }
    return RC_OK;
}

int rc_create(rc_ctx **out, const rc_config *cfg) {
    if (!out || !cfg) return RC_ERR_NULL_ARG;
    *out = nullptr;
    if (cfg->ncascades < 1 || cfg->ncascades > RC_MAX_CASCADES || !(cfg->c0_interval > 0.f) ||
        !std::isfinite(cfg->c0_interval))
        return RC_ERR_BAD_VALUE;
    if (cfg->lambda_batch != 0 && cfg->lambda_batch != 1 && cfg->lambda_batch != 2 &&
        cfg->lambda_batch != 4 && cfg->lambda_batch != 8)
        return RC_ERR_BAD_VALUE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) {
        cudaGetLastError();
        return RC_ERR_NO_DEVICE;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess || prop.major != 10)
        return RC_ERR_NO_DEVICE;  // sm_100a code only: no other backend, no fallback
    rc_ctx *ctx = new (std::nothrow) rc_ctx();
    if (!ctx) return RC_ERR_CUDA;
    ctx->cfg = *cfg;
    *out = ctx;
    return RC_OK;
}

int rc_destroy(rc_ctx *ctx) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (!ctx->ev.empty() || ctx->graph_exec || ctx->cap_stream || ctx->copy_stream) cudaSetDevice(ctx->cfg.device);
    for (auto &e : ctx->ev) cudaEventDestroy(e);
    if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    if (ctx->copy_stream) {
        cudaStreamDestroy(ctx->copy_stream);
        for (auto &e : ctx->pipe_ev) if (e) cudaEventDestroy(e);
    }
    delete ctx;
    return RC_OK;
}

// Where rc_solve_J_line_host stages the line parameters and J: in the host_io region of the GivenFs plan (which
// rc_workspace_bytes sizes), but never below the end of what the LINE plan's solve reads and writes - the two plans are
// laid out independently.  Returns the bytes of workspace this needs.
static size_t line_host_io_layout(const rc_ctx *ctx, int nx, int ny, int nlambda, size_t *o_line, size_t *o_J) {
    Plan Pio, Pl;
    make_plan(ctx->cfg, ctx->tune, ctx->nm, false, nx, ny, nlambda, true, Pio, nullptr);
    make_plan(ctx->cfg, ctx->tune, ctx->nm, true, nx, ny, nlambda, false, Pl, nullptr);
    const size_t ncell = (size_t)nx * ny;
    const size_t nout = ncell * ((ctx->cfg.flags & RC_ACCUM_J) ? 1 : (size_t)nlambda) * sizeof(float);
    *o_line = std::max(Pio.io_chi, align_up(Pl.total));
    *o_J = std::max(Pio.io_J, *o_line + align_up(ncell * 6 * sizeof(float)));
    return *o_J + align_up(nout);
}

size_t rc_workspace_bytes(const rc_ctx *ctx, int nx, int ny, int nlambda, int host_io) {
    if (!ctx) return 0;
    Plan P;
    if (!make_plan(ctx->cfg, ctx->tune, ctx->nm, false, nx, ny, nlambda, host_io != 0, P, nullptr)) return 0;
    size_t need = P.total;
    if (make_plan(ctx->cfg, ctx->tune, ctx->nm, true, nx, ny, nlambda, false, P, nullptr)) need = std::max(need, P.total);  // line mode
    if (host_io) {
        size_t a, b;
        need = std::max(need, line_host_io_layout(ctx, nx, ny, nlambda, &a, &b));  // rc_solve_J_line_host
    }
    return need;
}

int rc_set_workspace(rc_ctx *ctx, void *dev_ptr, size_t bytes) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (!dev_ptr || ((uintptr_t)dev_ptr % ALIGN) != 0)
        return fail(ctx, RC_ERR_NO_WORKSPACE, "workspace pointer is null or not %zu-byte aligned", ALIGN);
    ctx->ws = (char *)dev_ptr;
    ctx->ws_bytes = bytes;
    ctx->tab_nx = ctx->tab_ny = 0;  // tables live in the workspace: rebuild
    ctx->have_atm = false;
    ctx->xl_on_device = false;
    return RC_OK;
}

int rc_set_stream(rc_ctx *ctx, void *cuda_stream) {
    if (!ctx) return RC_ERR_NULL_ARG;
    ctx->stream = (cudaStream_t)cuda_stream;
    return RC_OK;
}

int rc_set_tuning(rc_ctx *ctx, const char *name, double value) {
    if (!ctx || !name) return RC_ERR_NULL_ARG;
    Tuning &t = ctx->tune;
    const std::string n(name);
    const int iv = (int)std::lround(value);
    if (n == "march_variant") { if (iv < -1 || iv > 4) goto bad; t.variant = iv; }
    else if (n == "patch_log2") { if (iv != -1 && (iv < 2 || iv > 5)) goto bad; t.patch_log2 = iv; }
    else if (n == "patch_from") { if (iv < 0) goto bad; t.patch_from = iv; }
    else if (n == "cpw_from") { if (iv < -1) goto bad; t.cpw_from = iv; t.cpw_forced = true; }
    else if (n == "tau_cut") { if (!(value >= 1.0)) goto bad; t.tau_cut = (float)value; }
    else if (n == "bands") { if (iv < 0) goto bad; t.bands = iv; }
    else if (n == "l2_mb") { if (!(value >= 1.0)) goto bad; t.l2_mb = value; }
    else if (n == "sparse") { if (iv < -1 || iv > 1) goto bad; t.sparse = iv; }
    else if (n == "graph") { t.graph = iv != 0; }
    else if (n == "sparse_mode") { if (iv < 0 || iv > 3) goto bad; t.sparse_mode = iv; }
    else if (n == "lists") { t.lists = iv != 0; }
    else if (n == "pipeline") { t.pipeline = iv != 0; }
    else if (n == "list_b") { if (iv != 0 && iv != 1 && iv != 2 && iv != 4 && iv != 8) goto bad; t.list_b = iv; }
    else if (n == "sorted") { if (iv < -1 || iv > 1) goto bad; t.sorted = iv; }
    else return fail(ctx, RC_ERR_BAD_VALUE, "rc_set_tuning: unknown knob '%s'", name);
    // the plan (bands), the patch lists and a captured graph may depend on a knob: start over
    ctx->tune_gen++;
    ctx->have_atm = false;
    ctx->active_set = false; ctx->lists_dirty = false; ctx->sparse = false; ctx->lists_built = false;
    return RC_OK;
bad:
    return fail(ctx, RC_ERR_BAD_VALUE, "rc_set_tuning: %s = %g is out of range", name, value);
}

int rc_set_timing(rc_ctx *ctx, int nsets) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (nsets < 0 || nsets > 4096) return fail(ctx, RC_ERR_BAD_VALUE, "nsets must be in [0, 4096]");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    for (auto &e : ctx->ev) cudaEventDestroy(e);
    ctx->ev.clear();
    const int per = 2 * ctx->cfg.ncascades + 2;
    ctx->ev.resize((size_t)nsets * per);
    for (auto &e : ctx->ev) RC_CUDA(ctx, cudaEventCreate(&e));
    ctx->nsets = nsets;
    ctx->solves_timed = 0;
    return RC_OK;
}

// Plan, step tables and defaults for a shape (shared by rc_set_atmosphere and rc_set_line_atmosphere).
static int prepare_shape(rc_ctx *ctx, int nx, int ny, int nlambda, bool line) {
    if (!shape_ok(ctx->cfg, nx, ny, nlambda))
        return fail(ctx, RC_ERR_BAD_SHAPE, "nx=%d ny=%d nlambda=%d: need positive multiples of 2^(ncascades-1)=%d, <= %d",
                    nx, ny, nlambda, 1 << (ctx->cfg.ncascades - 1), RC_MAX_DIM);
    if (!ctx->ws) return fail(ctx, RC_ERR_NO_WORKSPACE, "rc_set_workspace has not been called");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const bool same_shape = ctx->have_atm && ctx->plan.nx == nx && ctx->plan.ny == ny && ctx->plan.L == nlambda && ctx->plan.line == line;
    if (!same_shape) {
        Plan P, Pio;
        std::vector<std::vector<long long>> offs;
        make_plan(ctx->cfg, ctx->tune, ctx->nm, line, nx, ny, nlambda, false, P, &offs);
        if (P.total > ctx->ws_bytes)
            return fail(ctx, RC_ERR_NO_WORKSPACE, "workspace has %zu bytes, %zu needed", ctx->ws_bytes, P.total);
        make_plan(ctx->cfg, ctx->tune, ctx->nm, line, nx, ny, nlambda, true, Pio, nullptr);
        ctx->host_io = Pio.total <= ctx->ws_bytes;
        ctx->plan = ctx->host_io ? Pio : P;
        ctx->have_atm = false;
        ctx->xl_on_device = false;  // plan.xls depends on the shape and the banding
        ctx->active_set = false; ctx->lists_dirty = false; ctx->sparse = false; ctx->lists_built = false;
        ctx->stats.active_cells = -1;
        // geometry tables: only when the grid size changed (they do not depend on nlambda)
        if (ctx->tab_nx != nx || ctx->tab_ny != ny) {
            ctx->off_host.swap(offs);
            const int top = ctx->cfg.ncascades - 1;
            for (int i = 0; i <= top; i++) {
                const CascadePlan &c = ctx->plan.c[i];
                ctx->stats.table_steps[i] = c.slots;
                if (c.empty) continue;
                RC_CUDA(ctx, cudaMemcpyAsync(ctx->ws + c.off_off, ctx->off_host[i].data(),
                                             sizeof(long long) * ctx->off_host[i].size(), cudaMemcpyHostToDevice, ctx->stream));
                rc::TableBuildParams tp;
                tp.steps = (rc::Step *)(ctx->ws + c.steps_off);
                tp.xy = (rc::StepXY *)(ctx->ws + c.xy_off);
                tp.off = (const long long *)(ctx->ws + c.off_off);
                tp.cnt = (int *)(ctx->ws + c.cnt_off);
                tp.cascade = i; tp.top = i == top; tp.ndir = c.ndir;
                tp.ta = c.ta; tp.tb = c.tb; tp.nx = nx; tp.ny = ny;
                tp.fix = c.fix; tp.subdir = c.fix ? (float2 *)(ctx->ws + c.subdir_off) : nullptr;
                RC_CUDA(ctx, rc::launch_table_build(tp, ctx->stream));
            }
            ctx->tab_nx = nx; ctx->tab_ny = ny;
        }
        // sorted quad lists (they depend on the plan: banding, the fix - not only on the grid size)
        ctx->qlist_host.assign(ctx->cfg.ncascades, {});
        for (int i = 0; i < ctx->cfg.ncascades; i++) {
            const CascadePlan &c = ctx->plan.c[i];
            if (!c.sorted) continue;
            sorted_quads(nx, ny, i, c.ta, c.tb, c.qpad, &ctx->qlist_host[i], c.fix ? 2 : 1);
            RC_CUDA(ctx, cudaMemcpyAsync(ctx->ws + c.qlist_off, ctx->qlist_host[i].data(), sizeof(unsigned short) * ctx->qlist_host[i].size(),
                                         cudaMemcpyHostToDevice, ctx->stream));
        }
        // defaults: free-space boundary, unit weights
        ctx->stage.assign((size_t)ctx->plan.Lpad, 0.f);
        RC_CUDA(ctx, cudaMemsetAsync(ctx->ws + ctx->plan.bc_below, 0, (size_t)ctx->plan.Lpad * ctx->plan.NM * sizeof(float), ctx->stream));
        RC_CUDA(ctx, cudaMemsetAsync(ctx->ws + ctx->plan.bc_above, 0, (size_t)ctx->plan.Lpad * ctx->plan.NM * sizeof(float), ctx->stream));
        std::vector<float> ones((size_t)ctx->plan.Lpad, 0.f);
        for (int l = 0; l < nlambda; l++) ones[l] = 1.f;
        RC_CUDA(ctx, cudaMemcpyAsync(ctx->ws + ctx->plan.weights, ones.data(), ones.size() * sizeof(float),
                                     cudaMemcpyHostToDevice, ctx->stream));
        RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));  // `ones` and the offsets are host temporaries
    }
    return RC_OK;
}

// The kernels read and write the caller's arrays with 32-byte vector accesses (one sector per thread).
static bool aligned32(const void *p) { return ((uintptr_t)p & 31) == 0; }

int rc_set_atmosphere(rc_ctx *ctx, const float *chi, const float *eta, int nx, int ny, int nlambda) {
    if (!ctx || !chi || !eta) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null chi/eta") : RC_ERR_NULL_ARG;
    if (!aligned32(chi) || !aligned32(eta)) return fail(ctx, RC_ERR_BAD_VALUE, "chi and eta must be 32-byte aligned");
    {
        const int rc = prepare_shape(ctx, nx, ny, nlambda, false);
        if (rc != RC_OK) return rc;
    }
    ctx->line = nullptr;
    ctx->xl_on_device = false;
    if (ctx->cfg.flags & RC_VALIDATE) {
        int *flag = (int *)(ctx->ws + ctx->plan.flag);
        int h = 0;
        RC_CUDA(ctx, cudaMemsetAsync(flag, 0, sizeof(int), ctx->stream));
        RC_CUDA(ctx, rc::launch_validate(chi, eta, (long long)nx * ny * nlambda, flag, ctx->stream));
        RC_CUDA(ctx, cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (h & 1) return fail(ctx, RC_ERR_BAD_VALUE, "chi or eta has a negative or non-finite value");
    }
    ctx->sparse = false;  // the distance field belongs to the atmosphere it was built from: rc_analyse_atmosphere again
    ctx->stats.sparse_march = 0;
    ctx->chi = chi;
    ctx->eta = eta;
    ctx->have_atm = true;
    return RC_OK;
}

// Velocity-dependent line mode.
int rc_set_line_atmosphere(rc_ctx *ctx, const float *line, int nx, int ny, const float *x_lambda, int nlambda) {
    if (!ctx || !line || !x_lambda) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null line / x_lambda") : RC_ERR_NULL_ARG;
    if (!aligned32(line)) return fail(ctx, RC_ERR_BAD_VALUE, "line must be 32-byte aligned");
    {
        const int rc = prepare_shape(ctx, nx, ny, nlambda, true);
        if (rc != RC_OK) return rc;
    }
    for (int l = 0; l < nlambda; l++)
        if (!std::isfinite(x_lambda[l])) return fail(ctx, RC_ERR_BAD_VALUE, "x_lambda[%d] is not finite", l);
    std::vector<float> h((size_t)2 * ctx->plan.Lpad, 0.f);
    for (int l = 0; l < nlambda; l++) {
        h[l] = (float)((double)x_lambda[l] * 1.2011224087864498);  // sqrt(log2 e)
        h[(size_t)ctx->plan.Lpad + l] = x_lambda[l];
    }
    if (!ctx->xl_on_device || h != ctx->xl_stage) {  // steady state (same wavelengths, same place): nothing to upload, nothing to wait for
        RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));  // an earlier upload may still be reading xl_stage
        ctx->xl_stage.swap(h);
        RC_CUDA(ctx, cudaMemcpyAsync(ctx->ws + ctx->plan.xls, ctx->xl_stage.data(), ctx->xl_stage.size() * sizeof(float),
                                     cudaMemcpyHostToDevice, ctx->stream));
        ctx->xl_on_device = true;
    }
    ctx->line = line;
    ctx->chi = ctx->eta = nullptr;
    ctx->sparse = false;
    ctx->have_atm = true;
    return RC_OK;
}

static int upload_lambda_array(rc_ctx *ctx, const float *src, size_t dst_off, float fill) {
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    std::vector<float> h((size_t)ctx->plan.Lpad, 0.f);
    for (int l = 0; l < ctx->plan.L; l++) h[l] = src ? src[l] : fill;
    RC_CUDA(ctx, cudaMemcpyAsync(ctx->ws + dst_off, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return RC_OK;
}

// Boundary arrays on the device are [Lpad][NM] (channel order).  per_inclination: src is [NM][L], else [L].
static int upload_boundary(rc_ctx *ctx, const float *src, size_t dst_off, bool per_inclination) {
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const int NM = ctx->plan.NM, L = ctx->plan.L;
    std::vector<float> h((size_t)ctx->plan.Lpad * NM, 0.f);
    for (int l = 0; l < L && src; l++)
        for (int m = 0; m < NM; m++) {
            const float v = per_inclination ? src[(size_t)m * L + l] : src[l];
            if (!(v >= 0.f) || !std::isfinite(v)) return fail(ctx, RC_ERR_BAD_VALUE, "boundary intensity must be finite and >= 0");
            h[(size_t)l * NM + m] = v;
        }
    RC_CUDA(ctx, cudaMemcpyAsync(ctx->ws + dst_off, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return RC_OK;
}

static int set_boundary_impl(rc_ctx *ctx, const float *I_below, const float *I_above, bool per_inclination) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    int rc = upload_boundary(ctx, I_below, ctx->plan.bc_below, per_inclination);
    if (rc != RC_OK) return rc;
    rc = upload_boundary(ctx, I_above, ctx->plan.bc_above, per_inclination);
    return rc;
}

int rc_set_boundary(rc_ctx *ctx, const float *I_below, const float *I_above) { return set_boundary_impl(ctx, I_below, I_above, false); }

int rc_set_boundary_inclined(rc_ctx *ctx, const float *I_below, const float *I_above) { return set_boundary_impl(ctx, I_below, I_above, true); }

// 2.5D: every flatland ray becomes n rays with the same projection and direction cosine mu[m] to the
// invariant axis; changes the workspace plan, so the atmosphere must be set again.
int rc_set_inclinations(rc_ctx *ctx, int n, const float *mu, const float *w) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (n != 1 && n != 2 && n != 4 && n != 8) return fail(ctx, RC_ERR_BAD_VALUE, "n = %d inclinations: must be 1, 2, 4 or 8", n);
    if ((!mu || !w) && n != 1) return fail(ctx, RC_ERR_NULL_ARG, "null mu / w");
    for (int m = 0; m < n && mu && w; m++)
        if (!(mu[m] >= 0.f) || !(mu[m] < 1.f) || !(w[m] >= 0.f) || !std::isfinite(w[m]))
            return fail(ctx, RC_ERR_BAD_VALUE, "inclination %d: need 0 <= mu < 1 and a finite weight >= 0", m);
    ctx->nm = n;
    for (int m = 0; m < 8; m++) {
        const bool on = m < n && mu && w;
        ctx->incl_f[m] = on ? (float)(1.0 / std::sqrt(1.0 - (double)mu[m] * (double)mu[m])) : 1.f;
        ctx->incl_w[m] = on ? w[m] : (m == 0 ? 1.f : 0.f);
    }
    ctx->have_atm = false;  // the plan (channels per lane, cascade storage) depends on n
    return RC_OK;
}

int rc_set_lambda_weights(rc_ctx *ctx, const float *w) {
    if (!ctx) return RC_ERR_NULL_ARG;
    return upload_lambda_array(ctx, w, ctx->plan.weights, 1.f);
}

// Register-ring depth / occupancy variant of cascade i's march launch (rc_kernels.cu, launch_march_flat): measured
// on config 2, short rays (cascades <= 3) like 20 warps/SM with a ring of 2, long rays 16 warps/SM with a ring of 3.
static int march_variant(const rc_ctx *ctx, int i) { return ctx->tune.variant >= 0 ? ctx->tune.variant : (i <= 3 ? 4 : 2); }

// Under the march over hit lists: does cascade i use them (else it runs lock-step)?
// (moving line: from cascade 1 - measured on the paper's regime, cascade 1: 8.2 ms over lists, 13.1 ms lock-step)
static bool list_cascade(const rc_ctx *ctx, int i) { return i >= (ctx->line ? 1 : 2) && !ctx->plan.c[i].empty; }

// Parameters of cascade i's march launch.
static rc::MarchParams march_params(const rc_ctx *ctx, int i, float *J_out) {
    const Plan &P = ctx->plan;
    const CascadePlan &c = P.c[i];
    const int top = ctx->cfg.ncascades - 1;
    const bool accum = (ctx->cfg.flags & RC_ACCUM_J) != 0;
    rc::MarchParams mp;
    const bool multi = P.multi_pack && !ctx->sparse && !ctx->line && !c.empty;
    mp.chiT = (const float *)(ctx->ws + (multi ? P.chiT_c[i] : P.chiT));
    mp.ST = (const float *)(ctx->ws + (multi ? P.ST_c[i] : P.ST));
    mp.linepk = ctx->line ? (const float *)(ctx->ws + P.chiT) : nullptr;
    mp.xls = ctx->line ? (const float *)(ctx->ws + P.xls) : nullptr;
    mp.dist = ctx->sparse ? (const unsigned char *)(ctx->ws + P.dist) : nullptr;
    mp.sparse_mode = ctx->tune.sparse_mode;
    // over hit lists from cascade 2 up; cascades 0 and 1 (rays of a few steps: nothing to skip, the merge is the work) and
    // cascades outside the box (boundary term and merge only) run lock-step even then (config 4: 24 of 134 ms -> 15)
    const bool lists = ctx->sparse && ctx->lists && list_cascade(ctx, i);
    if (ctx->sparse && ctx->lists && !lists) mp.dist = nullptr;
    mp.hit_off = lists ? (const unsigned *)(ctx->sws + ctx->hit_off[i]) : nullptr;
    mp.hit_list = lists ? (const unsigned short *)(ctx->sws + ctx->hit_list[i]) : nullptr;
    mp.list_b = ctx->list_b;
    mp.walked = ctx->count_walked ? (unsigned long long *)(ctx->ws + P.flag) + 16 + i : nullptr;
    mp.flags = ctx->active_set ? (const unsigned char *)(ctx->ws + P.pflag[i]) : nullptr;
    mp.plist = ctx->active_set && !ctx->lists_dirty ? (const int *)(ctx->ws + P.plist[i]) : nullptr;
    mp.npatch_act = ctx->npatch_act[i];
    mp.Aup = i == top ? nullptr : (const float *)(ctx->ws + P.A[(i + 1) & 1]);
    mp.out = i > 0 ? (float *)(ctx->ws + P.A[i & 1]) : (accum ? (float *)(ctx->ws + P.Jpart) : J_out);
    mp.steps = c.empty ? nullptr : (const rc::Step *)(ctx->ws + c.steps_off);
    mp.xy = c.empty ? nullptr : (const rc::StepXY *)(ctx->ws + c.xy_off);
    mp.off = c.empty ? nullptr : (const long long *)(ctx->ws + c.off_off);
    mp.cnt = c.empty ? nullptr : (const int *)(ctx->ws + c.cnt_off);
    mp.I_below = (const float *)(ctx->ws + P.bc_below);
    mp.I_above = (const float *)(ctx->ws + P.bc_above);
    mp.weights = (const float *)(ctx->ws + P.weights);
    mp.nx = P.nx; mp.ny = P.ny; mp.L = P.L; mp.nb = P.nb; mp.nb0 = 0;
    mp.cascade = i; mp.shift = i;
    mp.npx = P.nx >> i; mp.npy = P.ny >> i;
    mp.ngroups = 1 << (2 * i);
    mp.mode = i > 0 ? 0 : (accum ? 2 : 1);
    mp.early_exit = (ctx->cfg.flags & RC_NO_EARLY_EXIT) ? 0 : 1;
    mp.tau_cut = ctx->tune.tau_cut;
    mp.pw_log2 = ctx->tune.patch_log2 >= 0 && i >= ctx->tune.patch_from ? ctx->tune.patch_log2 : c.pw_log2;
    mp.fix = c.fix && !c.empty;
    mp.subdir = mp.fix ? (const float2 *)(ctx->ws + c.subdir_off) : nullptr;
    const int lx = mp.fix ? mp.npx >> 1 : mp.npx, ly = mp.fix ? mp.npy >> 1 : mp.npy;  // lane lattice
    while (mp.pw_log2 > 0 && (1 << mp.pw_log2) > lx) mp.pw_log2--;
    const int pw = 1 << mp.pw_log2, ph = 32 >> mp.pw_log2;
    mp.npatch_x = (lx + pw - 1) / pw;
    mp.npatch_y = (ly + ph - 1) / ph;
    mp.kg_n = mp.ngroups; mp.kg_off = 0;
    // sorted quads: dense, unbanded launches of the whole direction circle (not with flagged probes, whose compacted
    // patch lists number rectangular patches, and not under the distance-field march)
    const bool sorted = c.sorted && !ctx->active_set && !ctx->sparse;
    mp.qlist = sorted ? (const unsigned short *)(ctx->ws + c.qlist_off) : nullptr;
    mp.qpad = sorted ? c.qpad : 0;
    // child-per-warp where the march is bound by the L2 -> SM gathers (measured: config 2 77.0 -> 73.7 ms, config 3
    // 331 -> 315 ms, bilinear fix 341 -> 321 ms); not in the MUFU-bound modes (inclinations, moving line)
    // ... nor on a cascade that barely reaches into the box (config 2, cascade 6: 0.014 % of its rays are live)
    const double diag = std::sqrt((double)P.nx * P.nx + (double)P.ny * P.ny);
    const bool reaches = std::fmin(c.tb, diag) - c.ta > 0.2 * c.ta || i == 0;
    // ... and on every cascade of a small grid, which is bound by the serial chain of one warp's 4 children (config 0: 107 -> 89 us)
    const bool small = (long long)P.nx * P.ny * P.Lpad * P.NM <= (1LL << 21);
    const int cpw_from = small && !ctx->tune.cpw_forced ? 0 : ctx->tune.cpw_from;
    mp.cpw = J_out != nullptr && cpw_from >= 0 && i >= cpw_from && !c.empty && (reaches || ctx->tune.cpw_forced) && !ctx->sparse &&
             P.NM == 1 && !ctx->line ? 1 : 0;
    for (int m = 0; m < 8; m++) { mp.incl_f[m] = ctx->incl_f[m]; mp.incl_w[m] = ctx->incl_w[m]; mp.incl_s[m] = 1.f / ctx->incl_f[m]; }
    mp.state = nullptr;
    mp.band_axis = 0; mp.band_sign = 1; mp.band_lo = 0; mp.band_hi = 0; mp.band_final = 1;
    return mp;
}

// Compacted patch lists ("the radiance intervals are only computed for these flagged probes"): for every
// cascade the numbers of the patches - in the numbering of the march's own warp -> probe mapping - that hold a flagged
// probe.  Synchronises (the counts size the launches).
static int build_patch_lists(rc_ctx *ctx) {
    const Plan &P = ctx->plan;
    ctx->lists_dirty = true;  // march_params must describe the full patch grid while the lists are built
    int *cnt = (int *)(ctx->ws + P.pcount);
    for (int i = 0; i < ctx->cfg.ncascades; i++) {
        rc::MarchParams mp = march_params(ctx, i, nullptr);
        mp.nb = 1; mp.cpw = 0; mp.plist = nullptr;
        const long long npatch = (long long)mp.npatch_x * mp.npatch_y * (mp.fix ? 4 : 1);
        if (npatch > P.plist_cap[i]) return fail(ctx, RC_ERR_CUDA, "patch list of cascade %d: %lld > capacity %d", i, npatch, P.plist_cap[i]);
        RC_CUDA(ctx, rc::launch_mark_and_compact_patches(mp, (int)npatch, (unsigned char *)(ctx->ws + P.pmark), (int *)(ctx->ws + P.plist[i]),
                                                         cnt + i, ctx->stream));
    }
    int h[RC_MAX_CASCADES];
    RC_CUDA(ctx, cudaMemcpyAsync(h, cnt, sizeof(int) * ctx->cfg.ncascades, cudaMemcpyDeviceToHost, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < ctx->cfg.ncascades; i++) ctx->npatch_act[i] = h[i];
    ctx->lists_dirty = false;
    ctx->list_version++;
    return RC_OK;
}

// One full solve: for cascade i = top .. 0 { pack chi/eta for spacing 2^i ; march + merge }  (PAPER.md:207:
// "after calculation, each interval of cascade i merges with the child intervals of cascade i+1.
// Cascade i-1 is then computed and merged with cascade i").
// b0, bn: the wavelength batches to solve (default: all of them); wavelengths are independent, so
// rc_solve_J_host solves them in two halves while the other half's copies are in flight.
static int enqueue_solve(rc_ctx *ctx, float *J_out, int b0 = 0, int bn = -1) {
    const Plan &P = ctx->plan;
    if (bn < 0) bn = P.nb;
    const bool whole = b0 == 0 && bn == P.nb, last = b0 + bn == P.nb;
    const int top = ctx->cfg.ncascades - 1;
    const bool accum = (ctx->cfg.flags & RC_ACCUM_J) != 0;
    const int per = 2 * ctx->cfg.ncascades + 2;
    cudaEvent_t *ev = ctx->nsets > 0 && whole ? ctx->ev.data() + (size_t)(ctx->solves_timed % ctx->nsets) * per : nullptr;
    int launches = whole || b0 == 0 ? 0 : ctx->stats.kernel_launches;
    if (ev) RC_CUDA(ctx, cudaEventRecord(ev[0], ctx->stream));
    if (ctx->active_set && b0 == 0) {
        // J is computed on the cells of interest only: the others read 0
        const size_t ncell = (size_t)P.nx * P.ny;
        if (accum) RC_CUDA(ctx, cudaMemsetAsync(ctx->ws + P.Jpart, 0, ncell * P.nb * sizeof(float), ctx->stream));
        else RC_CUDA(ctx, cudaMemsetAsync(J_out, 0, ncell * P.L * sizeof(float), ctx->stream));
    }
    auto pack = [&](int shift, bool list_layout = true) -> int {
        rc::PackParams pp{};
        pp.chi = ctx->chi; pp.eta = ctx->eta;
        pp.chiT = (float *)(ctx->ws + P.chiT); pp.ST = (float *)(ctx->ws + P.ST);
        pp.active = ctx->active_set ? (const unsigned char *)(ctx->ws + P.pflag[0]) : nullptr;
        pp.nx = P.nx; pp.ny = P.ny; pp.L = P.L; pp.nb = bn; pp.nb0 = b0; pp.shift = shift;
        // thin form below chi ds log2e = 1/64 for the longest segment (sqrt2 cells) of the most inclined ray, roughly:
        // there the trapezoid is good to 2e-5 (seg_update*() in rc_kernels.cu)
        float fmax = 1.f;
        for (int m = 0; m < ctx->nm; m++) fmax = std::max(fmax, ctx->incl_f[m]);
        pp.c_thin = (1.f / 64.f) / fmax;
        pp.list_b = ctx->sparse && ctx->lists && list_layout ? ctx->list_b : 0;
        if (ctx->line) {
            pp.chi = ctx->line; pp.eta = nullptr;
            RC_CUDA(ctx, rc::launch_pack_line(pp, ctx->stream));
        } else {
            RC_CUDA(ctx, rc::launch_pack(pp, P.LV, ctx->stream));
        }
        launches++;
        return RC_OK;
    };
    // the distance-field march gathers from plain cell order: one pack for every cascade
    if (ctx->sparse) { const int rc = pack(0); if (rc != RC_OK) return rc; }
    const bool multi = P.multi_pack && !ctx->sparse && !ctx->line;
    if (multi) {  // small grids: one launch packs for every cascade
        rc::PackParams pp{};
        pp.chi = ctx->chi; pp.eta = ctx->eta;
        pp.active = ctx->active_set ? (const unsigned char *)(ctx->ws + P.pflag[0]) : nullptr;
        pp.nx = P.nx; pp.ny = P.ny; pp.L = P.L; pp.nb = bn; pp.nb0 = b0;
        float fmax = 1.f;
        for (int m = 0; m < ctx->nm; m++) fmax = std::max(fmax, ctx->incl_f[m]);
        pp.c_thin = (1.f / 64.f) / fmax;
        pp.list_b = 0;
        for (int i = top; i >= 0; i--) {
            if (P.c[i].empty) continue;
            pp.shifts[pp.nmulti] = P.c[i].fix ? i + 1 : i;
            pp.chiTm[pp.nmulti] = (float *)(ctx->ws + P.chiT_c[i]);
            pp.STm[pp.nmulti] = (float *)(ctx->ws + P.ST_c[i]);
            pp.nmulti++;
        }
        if (pp.nmulti > 0) { RC_CUDA(ctx, rc::launch_pack(pp, P.LV, ctx->stream)); launches++; }
    }
    for (int i = top; i >= 0; i--) {
        const CascadePlan &c = P.c[i];
        if (!c.empty && !ctx->sparse && !multi) { const int rc = pack(c.fix ? i + 1 : i); if (rc != RC_OK) return rc; }
        // under the hit lists the lowest cascades run lock-step from their own phase-plane packing (the list cascades,
        // marched before them, are done with the packed arrays by then)
        if (!c.empty && ctx->sparse && ctx->lists && !list_cascade(ctx, i)) { const int rc = pack(i, false); if (rc != RC_OK) return rc; }
        if (ev) RC_CUDA(ctx, cudaEventRecord(ev[1 + 2 * (top - i)], ctx->stream));
        rc::MarchParams mp = march_params(ctx, i, J_out);
        mp.nb = bn; mp.nb0 = b0;
        if (!c.banded || ctx->sparse) {  // the distance-field march gathers occupied cells only: they fit L2
            RC_CUDA(ctx, rc::launch_march(mp, P.LV * P.NM, P.NM, march_variant(ctx, i), ctx->stream));
            launches++;
        } else {
            // rays heading up (right) cross the bands in ascending order, the others in descending order;
            // the last band of each half does the merge and writes the cascade
            const int n_axis = P.band_axis ? P.nx : P.ny, ext = (n_axis + P.nbands - 1) / P.nbands;
            mp.state = (float *)(ctx->ws + P.state);
            mp.band_axis = P.band_axis;
            mp.kg_n = mp.ngroups / 2;
            for (int h = 0; h < 2; h++) {
                mp.band_sign = h == 0 ? 1 : -1;
                // rows: sin(theta_k) > 0 for the first half of the circle; columns: cos > 0 for the quarter either side of k = 0
                mp.kg_off = P.band_axis ? (h == 0 ? mp.ngroups - mp.ngroups / 4 : mp.ngroups / 4) : (h == 0 ? 0 : mp.ngroups / 2);
                for (int bi = 0; bi < P.nbands; bi++) {
                    const int beta = h == 0 ? bi : P.nbands - 1 - bi;
                    mp.band_lo = beta * ext;
                    mp.band_hi = std::min(n_axis, (beta + 1) * ext);
                    mp.band_final = bi == P.nbands - 1;
                    RC_CUDA(ctx, rc::launch_march(mp, P.LV * P.NM, P.NM, march_variant(ctx, i), ctx->stream));
                    launches++;
                }
            }
        }
        if (ev) RC_CUDA(ctx, cudaEventRecord(ev[2 + 2 * (top - i)], ctx->stream));
    }
    if (accum && last) {
        RC_CUDA(ctx, rc::launch_reduce_jbar((const float *)(ctx->ws + P.Jpart), J_out, (long long)P.nx * P.ny, P.nb, ctx->stream));
        launches++;
    }
    if (ev) {
        RC_CUDA(ctx, cudaEventRecord(ev[per - 1], ctx->stream));
        ctx->solves_timed++;
    }
    ctx->stats.kernel_launches = launches;
    return RC_OK;
}

// Small grids are launch bound (config 0: 11 launches of a few microseconds each): their launch sequence is
// captured once into a CUDA graph (on a private stream, so the caller's stream may be the legacy default
// stream) and replayed into the caller's stream until anything the launches depend on changes.
int rc_solve_J(rc_ctx *ctx, float *J_out) {
    if (!ctx || !J_out) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null J_out") : RC_ERR_NULL_ARG;
    if (!aligned32(J_out)) return fail(ctx, RC_ERR_BAD_VALUE, "J_out must be 32-byte aligned");
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    if (ctx->lists_dirty) { const int rc = build_patch_lists(ctx); if (rc != RC_OK) return rc; }
    const Plan &P = ctx->plan;
    bool use_graph = ctx->nsets == 0 && (long long)P.nx * P.ny * P.Lpad * P.NM <= (1LL << 21) && ctx->tune.graph != 0;
    if (use_graph) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(ctx->stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
            cudaGetLastError();
            use_graph = false;  // the caller is capturing us: just enqueue
        }
    }
    if (!use_graph) return enqueue_solve(ctx, J_out);
    rc_ctx::GraphKey key;
    std::memset(&key, 0, sizeof(key));
    key.J = J_out; key.chi = ctx->chi; key.eta = ctx->eta; key.line = ctx->line; key.ws = ctx->ws;
    key.nx = P.nx; key.ny = P.ny; key.L = P.L; key.nm = P.NM; key.sparse = (ctx->sparse ? 1 : 0) + (ctx->active_set ? 2 : 0) + 4 * ctx->list_version;  // (list_version also counts the analyses)
    key.total = P.total;
    key.tune_gen = ctx->tune_gen;
    for (int m = 0; m < 8; m++) { key.f[m] = ctx->incl_f[m]; key.w[m] = ctx->incl_w[m]; }
    if (!ctx->graph_exec || std::memcmp(&key, &ctx->graph_key, sizeof(key)) != 0) {
        if (ctx->graph_exec) { cudaGraphExecDestroy(ctx->graph_exec); ctx->graph_exec = nullptr; }
        if (!ctx->cap_stream) RC_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
        cudaStream_t user = ctx->stream;
        ctx->stream = ctx->cap_stream;
        cudaGraph_t g = nullptr;
        cudaError_t e = cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal);
        int rc = e == cudaSuccess ? enqueue_solve(ctx, J_out) : RC_ERR_CUDA;
        cudaError_t e2 = e == cudaSuccess ? cudaStreamEndCapture(ctx->cap_stream, &g) : e;
        ctx->stream = user;
        if (rc == RC_OK && e2 == cudaSuccess && g) e2 = cudaGraphInstantiate(&ctx->graph_exec, g, 0);
        if (g) cudaGraphDestroy(g);
        if (rc != RC_OK || e2 != cudaSuccess || !ctx->graph_exec) {
            cudaGetLastError();
            ctx->graph_exec = nullptr;
            return enqueue_solve(ctx, J_out);  // no graph: plain launches
        }
        ctx->graph_key = key;
    }
    RC_CUDA(ctx, cudaGraphLaunch(ctx->graph_exec, ctx->stream));
    return RC_OK;
}

// Sparsity as the paper defines it.
int rc_set_active_cells(rc_ctx *ctx, const unsigned char *active) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const Plan &P = ctx->plan;
    ctx->sparse = false;  // the distance field depends on the flags
    ctx->lists_built = false;
    if (!active) {
        ctx->active_set = false; ctx->lists_dirty = false;
        ctx->stats.active_cells = -1;
        ctx->list_version++;
        return RC_OK;
    }
    const int top = ctx->cfg.ncascades - 1;
    RC_CUDA(ctx, rc::launch_flags_from_active(active, (unsigned char *)(ctx->ws + P.pflag[0]), (long long)P.nx * P.ny, ctx->stream));
    for (int i = 0; i < top; i++) {
        RC_CUDA(ctx, cudaMemsetAsync(ctx->ws + P.pflag[i + 1], 0, (size_t)(P.nx >> (i + 1)) * (P.ny >> (i + 1)), ctx->stream));
        RC_CUDA(ctx, rc::launch_flag_parents((const unsigned char *)(ctx->ws + P.pflag[i]), P.nx >> i, P.ny >> i,
                                             (unsigned char *)(ctx->ws + P.pflag[i + 1]), ctx->stream));
    }
    ctx->active_set = true;
    {
        const int rc = build_patch_lists(ctx);
        if (rc != RC_OK) { ctx->active_set = false; return rc; }
    }
    // flagged probes per cascade, for the statistics: counted on the device, one small copy back (counters [32..43] of P.flag)
    {
        unsigned long long *d = (unsigned long long *)(ctx->ws + P.flag) + 32, h[RC_MAX_CASCADES] = {0};
        RC_CUDA(ctx, cudaMemsetAsync(d, 0, sizeof(h), ctx->stream));
        for (int i = 0; i <= top; i++)
            RC_CUDA(ctx, rc::launch_count_flags((const unsigned char *)(ctx->ws + P.pflag[i]), (long long)(P.nx >> i) * (P.ny >> i), d + i, ctx->stream));
        RC_CUDA(ctx, cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
        RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        for (int i = 0; i <= top; i++) ctx->stats.probes_flagged[i] = (int64_t)h[i];
    }
    ctx->stats.active_cells = ctx->stats.probes_flagged[0];
    return RC_OK;
}

// Hit lists of the sparse march (rc_kernels.cu "Hit lists"): per cascade the occupied in-box steps of every ray, found once
// per analysed atmosphere instead of once per wavelength batch and solve.  They live in the caller's second buffer
// (rc_set_sparse_workspace); how much they need is only known after counting, so the count always runs and
// rc_stats.sparse_list_bytes reports it - when the buffer is missing or too small the distance-field march stays in use.
static int build_hit_lists(rc_ctx *ctx) {
    const Plan &P = ctx->plan;
    const int nc = ctx->cfg.ncascades;
    const size_t nrays = 4 * (size_t)P.nx * P.ny;                 // per cascade
    const size_t off_bytes = align_up(sizeof(unsigned) * (nrays + 1));
    const size_t bsum_bytes = align_up(sizeof(unsigned) * ((nrays + 1023) / 1024 + 1));
    unsigned long long *tot_d = (unsigned long long *)(ctx->ws + P.flag);  // [0..15] scratch counters
    RC_CUDA(ctx, cudaMemsetAsync(tot_d, 0, sizeof(*tot_d) * 16, ctx->stream));
    // room for the offsets? then count per ray, else only the totals (to report the size)
    const size_t occ_bytes = align_up((size_t)P.nx * P.ny);      // the occupancy map the lists belong to
    size_t cur = occ_bytes + bsum_bytes;
    for (int i = 0; i < nc; i++) {
        if (!list_cascade(ctx, i)) continue;
        ctx->hit_off[i] = cur; cur += off_bytes;
    }
    const bool have_off = ctx->sws != nullptr && cur <= ctx->sws_bytes;
    for (int i = 0; i < nc; i++) {
        if (!list_cascade(ctx, i)) continue;
        rc::MarchParams mp = march_params(ctx, i, nullptr);
        RC_CUDA(ctx, rc::launch_hit_walk(mp, false, have_off ? (unsigned *)(ctx->sws + ctx->hit_off[i]) : nullptr, nullptr, tot_d + i, ctx->stream));
    }
    unsigned long long tot[16] = {0};
    RC_CUDA(ctx, cudaMemcpyAsync(tot, tot_d, sizeof(tot), cudaMemcpyDeviceToHost, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    bool fits32 = true;
    for (int i = 0; i < nc; i++) {
        if (!list_cascade(ctx, i)) continue;
        ctx->hit_list[i] = cur; cur += align_up(sizeof(unsigned short) * (size_t)tot[i] + 2);
        fits32 = fits32 && tot[i] < 0xffffffffULL;
    }
    ctx->stats.sparse_list_bytes = (int64_t)cur;
    ctx->list_bytes = (int64_t)cur;
    if (!have_off || cur > ctx->sws_bytes || !fits32) return RC_OK;  // no room (or too many hits): the distance-field march
    for (int i = 0; i < nc; i++) {
        if (!list_cascade(ctx, i)) continue;
        rc::MarchParams mp = march_params(ctx, i, nullptr);
        unsigned *off = (unsigned *)(ctx->sws + ctx->hit_off[i]);
        RC_CUDA(ctx, rc::launch_hit_scan(off, (long long)nrays, (unsigned *)(ctx->sws + occ_bytes), tot[i], ctx->stream));
        RC_CUDA(ctx, rc::launch_hit_walk(mp, true, off, (unsigned short *)(ctx->sws + ctx->hit_list[i]), nullptr, ctx->stream));
    }
    // Wavelength batches per warp: the lanes of a ray share its list and table reads (measured on config 4: 218 / 167 / 134
    // / 135 ms at 1 / 2 / 4 / 8 batches per warp; config 3 with 25 % of the cells flagged, 4 batches: 210 / 146 / 130 ms)
    ctx->list_b = ctx->tune.list_b > 0 ? ctx->tune.list_b : P.nb >= 6 ? 8 : P.nb >= 3 ? 4 : P.nb;
    RC_CUDA(ctx, cudaMemcpyAsync(ctx->sws, ctx->ws + P.occ8, (size_t)P.nx * P.ny, cudaMemcpyDeviceToDevice, ctx->stream));
    ctx->lists = true;
    ctx->lists_built = true;
    ctx->stats.sparse_lists = 1;
    return RC_OK;
}

// Free-space acceleration: occupancy and its distance transform for the current atmosphere and flags.
int rc_analyse_atmosphere(rc_ctx *ctx) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const Plan &P = ctx->plan;
    unsigned long long *cnt = (unsigned long long *)(ctx->ws + P.flag);
    unsigned long long h = 0;
    RC_CUDA(ctx, rc::launch_build_distance_field(ctx->chi, ctx->eta, ctx->line,
                                                 ctx->active_set ? (const unsigned char *)(ctx->ws + P.pflag[0]) : nullptr, P.nx, P.ny, P.L,
                                                 (int *)(ctx->ws + P.A[0]), (unsigned char *)(ctx->ws + P.occ8), (unsigned char *)(ctx->ws + P.d1),
                                                 (unsigned char *)(ctx->ws + P.dist), cnt, ctx->stream));  // A[0] is free between solves
    // hit lists built for an earlier atmosphere of the same shape and flags stay good while the occupancy map is the same
    // (the formal solutions of an iteration, change chi and eta, not where they vanish)
    int differs = 1;
    int *dflag = (int *)(cnt + 1);
    if (ctx->lists_built) {
        RC_CUDA(ctx, cudaMemsetAsync(dflag, 0, sizeof(int), ctx->stream));
        RC_CUDA(ctx, rc::launch_occ_differs((const unsigned char *)(ctx->ws + P.occ8), (const unsigned char *)ctx->sws, (long long)P.nx * P.ny, dflag, ctx->stream));
        RC_CUDA(ctx, cudaMemcpyAsync(&differs, dflag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    }
    RC_CUDA(ctx, cudaMemcpyAsync(&h, cnt, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->stats.empty_cells = (int64_t)h;
    ctx->analysed = true;
    // the distance-field walk exists for the plain mode (no inclinations, no moving line, no bilinear fix); the march over
    // hit lists also with inclinations and the moving line (it then needs the lists: without the second buffer such a
    // solve stays lock-step)
    const bool can_list = !(ctx->cfg.flags & RC_BILINEAR_FIX);
    const bool can_walk = can_list && P.NM == 1 && !ctx->line;
    const bool want = ctx->tune.sparse >= 0 ? ctx->tune.sparse != 0 : 3 * h > 2ULL * P.nx * P.ny;
    ctx->sparse = want && (can_walk || (can_list && ctx->tune.lists != 0));
    ctx->stats.sparse_march = ctx->sparse;
    ctx->list_version++;
    ctx->lists = false;
    ctx->stats.sparse_lists = 0;
    ctx->stats.sparse_list_bytes = 0;
    if (ctx->sparse && ctx->tune.lists != 0) {
        if (ctx->lists_built && !differs) {
            ctx->lists = true;
            ctx->stats.sparse_lists = 2;
            ctx->stats.sparse_list_bytes = ctx->list_bytes;
        } else {
            ctx->lists_built = false;
            const int rc = build_hit_lists(ctx);
            if (rc != RC_OK) return rc;
        }
    }
    if (ctx->sparse && !ctx->lists && !can_walk) {  // inclined, and no room for the lists: the lock-step march
        ctx->sparse = false;
        ctx->stats.sparse_march = 0;
    }
    return RC_OK;
}

int rc_set_sparse_workspace(rc_ctx *ctx, void *dev_ptr, size_t bytes) {
    if (!ctx) return RC_ERR_NULL_ARG;
    if (dev_ptr && ((uintptr_t)dev_ptr % ALIGN) != 0) return fail(ctx, RC_ERR_NO_WORKSPACE, "sparse workspace pointer is not %zu-byte aligned", ALIGN);
    ctx->sws = (char *)dev_ptr;
    ctx->sws_bytes = dev_ptr ? bytes : 0;
    ctx->lists = false; ctx->lists_built = false;  // the lists lived in the old buffer: rc_analyse_atmosphere again
    ctx->list_version++;
    return RC_OK;
}

// Geometric segment count per cascade and wavelength (the unit of the throughput metric).
int rc_count_segments(rc_ctx *ctx, int64_t *per_cascade) {
    if (!ctx || !per_cascade) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null output") : RC_ERR_NULL_ARG;
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    unsigned long long *d = (unsigned long long *)(ctx->ws + ctx->plan.flag);
    RC_CUDA(ctx, cudaMemsetAsync(d, 0, ALIGN, ctx->stream));
    for (int i = 0; i < ctx->cfg.ncascades; i++)
        if (!ctx->plan.c[i].empty) RC_CUDA(ctx, rc::launch_count(march_params(ctx, i, nullptr), d + i, ctx->stream));
    unsigned long long h[RC_MAX_CASCADES];
    RC_CUDA(ctx, cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < ctx->cfg.ncascades; i++) per_cascade[i] = (int64_t)h[i];
    return RC_OK;
}

// One solve with counters: the cell segments the march integrated (early exit, sparsity and free-space jumps leave the
// rest out), per cascade, summed over the wavelength batches and divided by their number.
int rc_count_walked(rc_ctx *ctx, float *J_out, int64_t *per_cascade) {
    if (!ctx || !J_out || !per_cascade) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null argument") : RC_ERR_NULL_ARG;
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    if (ctx->lists_dirty) { const int rc = build_patch_lists(ctx); if (rc != RC_OK) return rc; }
    unsigned long long *d = (unsigned long long *)(ctx->ws + ctx->plan.flag) + 16;
    RC_CUDA(ctx, cudaMemsetAsync(d, 0, 16 * sizeof(*d), ctx->stream));
    ctx->count_walked = true;
    const int rc = enqueue_solve(ctx, J_out);
    ctx->count_walked = false;
    if (rc != RC_OK) return rc;
    unsigned long long h[16];
    RC_CUDA(ctx, cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < ctx->cfg.ncascades; i++) per_cascade[i] = (int64_t)(h[i] / (unsigned long long)ctx->plan.nb);
    return RC_OK;
}

// Line mode with HOST buffers: line_host [ny][nx][6], J_host as rc_solve_J_host.
int rc_solve_J_line_host(rc_ctx *ctx, const float *line_host, int nx, int ny, const float *x_lambda, int nlambda, float *J_host) {
    if (!ctx || !line_host || !x_lambda || !J_host) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null host buffer") : RC_ERR_NULL_ARG;
    if (!shape_ok(ctx->cfg, nx, ny, nlambda)) return fail(ctx, RC_ERR_BAD_SHAPE, "bad shape %dx%dx%d", nx, ny, nlambda);
    if (!ctx->ws) return fail(ctx, RC_ERR_NO_WORKSPACE, "rc_set_workspace has not been called");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    size_t o_line, o_J;
    const size_t need = line_host_io_layout(ctx, nx, ny, nlambda, &o_line, &o_J);
    if (need > ctx->ws_bytes)
        return fail(ctx, RC_ERR_NO_WORKSPACE, "workspace has %zu bytes, %zu needed with host_io", ctx->ws_bytes, need);
    const size_t nline = (size_t)nx * ny * 6 * sizeof(float);
    float *dline = (float *)(ctx->ws + o_line), *dJ = (float *)(ctx->ws + o_J);
    RC_CUDA(ctx, cudaMemcpyAsync(dline, line_host, nline, cudaMemcpyHostToDevice, ctx->stream));
    int rc = rc_set_line_atmosphere(ctx, dline, nx, ny, x_lambda, nlambda);
    if (rc != RC_OK) return rc;
    if (ctx->analysed) { rc = rc_analyse_atmosphere(ctx); if (rc != RC_OK) return rc; }
    rc = rc_solve_J(ctx, dJ);
    if (rc != RC_OK) return rc;
    const size_t nout = (size_t)nx * ny * ((ctx->cfg.flags & RC_ACCUM_J) ? 1 : nlambda) * sizeof(float);
    RC_CUDA(ctx, cudaMemcpyAsync(J_host, dJ, nout, cudaMemcpyDeviceToHost, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return RC_OK;
}

int rc_solve_J_host(rc_ctx *ctx, const float *chi_host, const float *eta_host, int nx, int ny,
                    int nlambda, float *J_host) {
    if (!ctx || !chi_host || !eta_host || !J_host) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null host buffer") : RC_ERR_NULL_ARG;
    if (!shape_ok(ctx->cfg, nx, ny, nlambda)) return fail(ctx, RC_ERR_BAD_SHAPE, "bad shape %dx%dx%d", nx, ny, nlambda);
    if (!ctx->ws) return fail(ctx, RC_ERR_NO_WORKSPACE, "rc_set_workspace has not been called");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    Plan Pio;
    make_plan(ctx->cfg, ctx->tune, ctx->nm, false, nx, ny, nlambda, true, Pio, nullptr);
    if (Pio.total > ctx->ws_bytes)
        return fail(ctx, RC_ERR_NO_WORKSPACE, "workspace has %zu bytes, %zu needed with host_io", ctx->ws_bytes, Pio.total);
    const size_t n = (size_t)nx * ny * nlambda * sizeof(float);
    float *dchi = (float *)(ctx->ws + Pio.io_chi), *deta = (float *)(ctx->ws + Pio.io_eta), *dJ = (float *)(ctx->ws + Pio.io_J);
    // Wavelengths are independent: large dense solves run as two halves of the wavelength batches, the
    // second half's inputs and the first half's J crossing PCIe (strided 2D copies on a private stream) while the other
    // half is solved.  Exposed: the first half's H2D and the second half's D2H instead of all of both.
    const size_t ncell = (size_t)nx * ny;
    // (not with RC_VALIDATE: the check reads the device copies, so they have to be complete before rc_set_atmosphere runs it)
    const bool pipelined = ctx->tune.pipeline != 0 && !ctx->analysed && ctx->nsets == 0 && !(ctx->cfg.flags & (RC_ACCUM_J | RC_VALIDATE)) &&
                           Pio.nb >= 2 && (long long)ncell * Pio.Lpad * Pio.NM >= (1LL << 24);  // (config 1, 4 M cell-channels: slower in halves)
    if (pipelined) {
        int rc = rc_set_atmosphere(ctx, dchi, deta, nx, ny, nlambda);  // pointers (and, for a new shape, the tables)
        if (rc != RC_OK) return rc;
        if (ctx->lists_dirty) { rc = build_patch_lists(ctx); if (rc != RC_OK) return rc; }
        if (!ctx->copy_stream) {
            RC_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
            for (auto &e : ctx->pipe_ev) RC_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        }
        const Plan &P = ctx->plan;
        cudaStream_t st = ctx->stream, cs = ctx->copy_stream;
        const int h = P.nb / 2;                                        // batches [0, h) and [h, nb)
        const size_t pitch = (size_t)nlambda * sizeof(float);
        const size_t col[3] = {0, (size_t)h * P.LV, (size_t)nlambda};  // their wavelength columns
        cudaEvent_t *e = ctx->pipe_ev;
        RC_CUDA(ctx, cudaEventRecord(e[0], st));
        RC_CUDA(ctx, cudaStreamWaitEvent(cs, e[0], 0));
        for (int g = 0; g < 2; g++) {
            const size_t w = (col[g + 1] - col[g]) * sizeof(float);
            RC_CUDA(ctx, cudaMemcpy2DAsync(dchi + col[g], pitch, chi_host + col[g], pitch, w, ncell, cudaMemcpyHostToDevice, cs));
            RC_CUDA(ctx, cudaMemcpy2DAsync(deta + col[g], pitch, eta_host + col[g], pitch, w, ncell, cudaMemcpyHostToDevice, cs));
            RC_CUDA(ctx, cudaEventRecord(e[1 + g], cs));
        }
        RC_CUDA(ctx, cudaStreamWaitEvent(st, e[1], 0));
        rc = enqueue_solve(ctx, dJ, 0, h);
        if (rc != RC_OK) return rc;
        RC_CUDA(ctx, cudaEventRecord(e[3], st));
        RC_CUDA(ctx, cudaStreamWaitEvent(st, e[2], 0));
        rc = enqueue_solve(ctx, dJ, h, P.nb - h);
        if (rc != RC_OK) return rc;
        RC_CUDA(ctx, cudaStreamWaitEvent(cs, e[3], 0));
        RC_CUDA(ctx, cudaMemcpy2DAsync(J_host + col[0], pitch, dJ + col[0], pitch, (col[1] - col[0]) * sizeof(float), ncell, cudaMemcpyDeviceToHost, cs));
        RC_CUDA(ctx, cudaEventRecord(e[4], cs));
        RC_CUDA(ctx, cudaMemcpy2DAsync(J_host + col[1], pitch, dJ + col[1], pitch, (col[2] - col[1]) * sizeof(float), ncell, cudaMemcpyDeviceToHost, st));
        RC_CUDA(ctx, cudaStreamWaitEvent(st, e[4], 0));
        RC_CUDA(ctx, cudaStreamSynchronize(st));
        return RC_OK;
    }
    RC_CUDA(ctx, cudaMemcpyAsync(dchi, chi_host, n, cudaMemcpyHostToDevice, ctx->stream));
    RC_CUDA(ctx, cudaMemcpyAsync(deta, eta_host, n, cudaMemcpyHostToDevice, ctx->stream));
    int rc = rc_set_atmosphere(ctx, dchi, deta, nx, ny, nlambda);
    if (rc != RC_OK) return rc;
    if (ctx->analysed) { rc = rc_analyse_atmosphere(ctx); if (rc != RC_OK) return rc; }
    rc = rc_solve_J(ctx, dJ);
    if (rc != RC_OK) return rc;
    const size_t nout = (ctx->cfg.flags & RC_ACCUM_J) ? (size_t)nx * ny * sizeof(float) : n;
    RC_CUDA(ctx, cudaMemcpyAsync(J_host, dJ, nout, cudaMemcpyDeviceToHost, ctx->stream));
    RC_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return RC_OK;
}

// Diagonal ALO of cascade 0 (eq. 17) for the current atmosphere and inclination set.
int rc_compute_alo(rc_ctx *ctx, float *alo_out) {
    if (!ctx || !alo_out) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null alo_out") : RC_ERR_NULL_ARG;
    if (!ctx->have_atm) return fail(ctx, RC_ERR_NO_ATMOSPHERE, "call rc_set_atmosphere first");
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    rc::AloParams ap;
    ap.chi = ctx->line ? nullptr : ctx->chi;
    ap.line = ctx->line;
    ap.xl = ctx->line ? (const float *)(ctx->ws + ctx->plan.xls) + ctx->plan.Lpad : nullptr;  // unscaled copy
    ap.out = alo_out;
    ap.ncell = (long long)ctx->plan.nx * ctx->plan.ny;
    ap.L = ctx->plan.L;
    ap.nm = ctx->nm;
    for (int m = 0; m < 8; m++) { ap.f[m] = ctx->incl_f[m]; ap.w[m] = ctx->incl_w[m]; }
    RC_CUDA(ctx, rc::launch_alo(ap, ctx->stream));
    return RC_OK;
}

// Achieved GB/s of the march's gather pattern alone over the first `mbytes` MB of the workspace:
// path 0 = LDG.256 (what the march uses), path 1 = TMA bulk copies into a shared-memory ring.
static int probe_bandwidth(rc_ctx *ctx, int mbytes, int path, double *gbs) {
    if (!ctx || !gbs) return ctx ? fail(ctx, RC_ERR_NULL_ARG, "null output") : RC_ERR_NULL_ARG;
    if (!ctx->ws) return fail(ctx, RC_ERR_NO_WORKSPACE, "rc_set_workspace has not been called");
    const size_t bytes = (size_t)mbytes << 20;
    if (mbytes < 1 || bytes + ALIGN > ctx->ws_bytes)
        return fail(ctx, RC_ERR_BAD_VALUE, "probe region of %d MB does not fit the workspace (%zu bytes)", mbytes, ctx->ws_bytes);
    RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaDeviceProp prop;
    RC_CUDA(ctx, cudaGetDeviceProperties(&prop, ctx->cfg.device));
    const int blocks = prop.multiProcessorCount * 6, iters = 2048;  // LDG path: 48 warps per SM
    float *sink = (float *)(ctx->ws + bytes);
    cudaEvent_t e0, e1;
    RC_CUDA(ctx, cudaEventCreate(&e0));
    RC_CUDA(ctx, cudaEventCreate(&e1));
    float best = 1e30f;
    long long moved = (long long)blocks * 8 * iters * 1024LL;
    for (int rep = 0; rep < 4; rep++) {  // the first pass also brings the region into L2
        RC_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        if (path == 0)
            RC_CUDA(ctx, rc::launch_gather_probe((const float *)ctx->ws, bytes / 32, iters, blocks, sink, ctx->stream));
        else
            RC_CUDA(ctx, rc::launch_bulk_probe((const float *)ctx->ws, bytes / 32, iters, prop.multiProcessorCount, sink, ctx->stream, &moved));
        RC_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        RC_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        RC_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *gbs = (double)moved / (best * 1e-3) / 1e9;
    return RC_OK;
}

int rc_probe_gather_bandwidth(rc_ctx *ctx, int mbytes, double *gbs) { return probe_bandwidth(ctx, mbytes, 0, gbs); }
int rc_probe_bulk_copy_bandwidth(rc_ctx *ctx, int mbytes, double *gbs) { return probe_bandwidth(ctx, mbytes, 1, gbs); }

int rc_get_stats(rc_ctx *ctx, rc_stats *out) {
    if (!ctx || !out) return RC_ERR_NULL_ARG;
    rc_stats &s = ctx->stats;
    s.ncascades = ctx->cfg.ncascades;
    s.lambda_batch = ctx->plan.LV;
    s.workspace_bytes = ctx->plan.total;
    const int top = ctx->cfg.ncascades - 1;
    for (int i = 0; i <= top; i++) { s.rays[i] = 4LL * ctx->plan.nx * ctx->plan.ny; s.ms_pack[i] = s.ms_march[i] = 0.f; }
    s.ms_total = 0.f;
    s.solves_timed = (int)std::min<long long>(ctx->solves_timed, ctx->nsets);
    if (s.solves_timed > 0) {
        RC_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
        const int per = 2 * ctx->cfg.ncascades + 2;
        for (int n = 0; n < s.solves_timed; n++) {
            cudaEvent_t *ev = ctx->ev.data() + (size_t)n * per;
            RC_CUDA(ctx, cudaEventSynchronize(ev[per - 1]));
            float ms;
            for (int i = top; i >= 0; i--) {
                RC_CUDA(ctx, cudaEventElapsedTime(&ms, ev[2 * (top - i)], ev[1 + 2 * (top - i)]));
                s.ms_pack[i] += ms;
                RC_CUDA(ctx, cudaEventElapsedTime(&ms, ev[1 + 2 * (top - i)], ev[2 + 2 * (top - i)]));
                s.ms_march[i] += ms;
            }
            RC_CUDA(ctx, cudaEventElapsedTime(&ms, ev[0], ev[per - 1]));
            s.ms_total += ms;
        }
        for (int i = 0; i <= top; i++) { s.ms_pack[i] /= s.solves_timed; s.ms_march[i] /= s.solves_timed; }
        s.ms_total /= s.solves_timed;
    }
    *out = s;
    return RC_OK;
}

}  // extern "C"
