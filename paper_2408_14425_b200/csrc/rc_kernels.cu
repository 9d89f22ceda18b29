// rc_kernels.cu — sm_100a kernels of the radiance-cascades hot path.
//
//   table_build_kernel  fp64 DDA of ONE ray per (cascade, direction), relative to the probe's lattice
//                       vertex.  All probes of a cascade sit at the same sub-cell position
//                       ((a+1/2) 2^i is an integer for i >= 1; a cell centre for i = 0),
//                       so every probe's ray in direction k is an integer translate of this one: the
//                       cells it crosses and the lengths inside them are shared.
//   pack_kernel         chi, eta [y][x][l]  ->  chi*log2(e), S = eta/chi in the probe-strided layout
//                       [batch][y mod s][x mod s][y div s][x div s][LV]: the cells that a patch of
//                       neighbouring probes of cascade i touches at the same step form a patch of
//                       the same shape in one phase plane (rows of contiguous 32-byte sectors).
//   march_kernel        a1 (eq. 16 along the interval) + a2 (boundary)
//                       + a3 (bilinear parents, mean of the 4 children, merge eq. 11,
//                       PAPER.md:149-157, 199-207) + a4 on cascade 0 (J), fused.
//                       One warp = a pw x ph patch of 32 probes x 1 direction group (4 child directions
//                       in turn) x LV wavelengths per lane; geometry is warp-uniform (no divergence from
//                       the DDA itself), radiance in fp32, I and T never leave registers.
//                       Template switches: NM inclinations per wavelength (2.5D), PD = depth
//                       of the register ring the gathers run ahead in, BANDED (grids larger than L2: one
//                       band of rows/columns per launch, ray state parked in between), LINE (opacity evaluated per ray
//                       from the projected velocity).  Run-time switch: the bilinear fix
//                       (4 sub-rays per interval, 16 tables per direction).
//   march_fan_kernel    the same for mostly empty atmospheres: lanes = a fan of adjacent directions,
//                       every lane walks its own ray and jumps over free space on a distance field.
//   pack_line_kernel, alo_kernel, reduce_jbar_kernel, validate / mark_occupied / count_* kernels: small
//                       elementwise or counting passes;  gather_probe_kernel, bulk_probe_kernel: the
//                       march's gather pattern alone, through LDG.256 and through TMA bulk copies, for
//                       the roofline (rc_probe_*_bandwidth).
#include "rc_internal.h"

#include <math_constants.h>

namespace rc {

static constexpr unsigned FULL = 0xffffffffu;
static constexpr int WARPS_PER_BLOCK = 8;

// ------------------------------------------------------------------------------------------------
// Geometry tables (fp64).  Restates PAPER.md:171-176 (shell [t_i, t_{i+1}]) and PAPER.md:314 (DDA).
// ------------------------------------------------------------------------------------------------
__global__ void table_build_kernel(TableBuildParams p) {
    // one thread per table: direction k, and with the bilinear fix (p.fix) one of the 16 sub-rays
    // (parity class of the probe x parent slot) of that direction
    const int nsub = p.fix ? 16 : 1;
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= p.ndir * nsub) return;
    const long long k = id / nsub;
    const int sub = (int)(id - k * nsub);
    Step *out = p.steps + p.off[id];
    StepXY *oxy = p.xy + p.off[id];
    const long long cap = p.off[id + 1] - p.off[id];
    const int s = 1 << p.cascade, half = s >> 1;
    // cell (vertex cell + (dx, dy)) in the packed layout [y mod S][x mod S][y div S][x div S], relative to the
    // lane's own entry of phase plane 0.  Plain: S = s, the entry is the probe's (b, a), the vertex cell sits at
    // (half, half) of its S x S block.  Bilinear fix: lanes are probes of one parity class (pa, pb), packed with
    // S = 2s (the parents' spacing), entry (b div 2, a div 2), vertex cell at (pa s + half, pb s + half).
    const int pa = (sub >> 2) & 1, pb = sub >> 3;
    const int shift = p.cascade + (p.fix ? 1 : 0), S = 1 << shift;
    const int npx = p.nx >> shift, npy = p.ny >> shift;
    const int offx = (p.fix ? pa * s : 0) + half, offy = (p.fix ? pb * s : 0) + half;
    auto emit = [&](int n, int dx, int dy, double ds) {
        const int tx = dx + offx, ty = dy + offy;
        const int phase = ((ty & (S - 1)) << shift) + (tx & (S - 1));
        out[n].delta = phase * (npx * npy) + (ty >> shift) * npx + (tx >> shift);
        out[n].ds = (float)ds;
        oxy[n].dx = (int16_t)dx;
        oxy[n].dy = (int16_t)dy;
    };
    if (p.fix) {
        // Bilinear fix: from the usual start p + t_i w to the start of the child cone on parent q,
        // P_q + t_(i+1) w.  P_q - P_p per axis: even probe index -1.5 s (slot 0), +0.5 s (slot 1); odd -0.5 s, +1.5 s.
        const int sa = sub & 1, sb = (sub >> 1) & 1;
        double wx, wy;
        sincospi(2.0 * ((double)k + 0.5) / (double)p.ndir, &wy, &wx);
        const double ox = (pa == 0 ? (sa ? 0.5 : -1.5) : (sa ? 1.5 : -0.5)) * s;
        const double oy = (pb == 0 ? (sb ? 0.5 : -1.5) : (sb ? 1.5 : -0.5)) * s;
        const double pc = p.cascade == 0 ? 0.5 : 0.0;  // probe position relative to the corner of its vertex cell
        const double x0 = pc + p.ta * wx, y0 = pc + p.ta * wy;
        double ux = ox + (p.tb - p.ta) * wx, uy = oy + (p.tb - p.ta) * wy;
        double len = sqrt(ux * ux + uy * uy);
        ux /= len; uy /= len;
        p.subdir[id] = make_float2((float)ux, (float)uy);
        // no ray from inside the box is still inside beyond this
        len = fmin(len, fmin(ux != 0.0 ? (double)p.nx / fabs(ux) : INFINITY, uy != 0.0 ? (double)p.ny / fabs(uy) : INFINITY) + 2.0 * s);
        int ix = (int)floor(x0), iy = (int)floor(y0);
        if ((double)ix == x0 && ux < 0.0) ix--;
        if ((double)iy == y0 && uy < 0.0) iy--;
        const int sx = ux > 0.0 ? 1 : -1, sy = uy > 0.0 ? 1 : -1;
        int gx = ux > 0.0 ? ix + 1 : ix, gy = uy > 0.0 ? iy + 1 : iy;
        double tmx = ux != 0.0 ? ((double)gx - x0) / ux : INFINITY, tmy = uy != 0.0 ? ((double)gy - y0) / uy : INFINITY;
        double t = 0.0;
        int n = 0;
        while (n < cap) {
            const double tn = fmin(fmin(tmx, tmy), len);
            const double ds = tn - t;
            if (ds > 0.0) emit(n++, ix, iy, ds);
            if (tn >= len) break;
            const bool stepx = tmx <= tmy, stepy = tmy <= tmx;  // a tie is a corner: step both
            if (stepx) { ix += sx; gx += sx; tmx = ((double)gx - x0) / ux; }
            if (stepy) { iy += sy; gy += sy; tmy = ((double)gy - y0) / uy; }
            t = tn;
        }
        p.cnt[id] = n;
        return;
    }
    int n = 0;
    if (p.cascade == 0) {
        // The 4 diagonals from a cell centre pass exactly through cell corners: closed form.
        // Cell m along the diagonal covers t in [sqrt2 (m-1/2), sqrt2 (m+1/2)], cut to [ta, tb].
        const int sx = (k == 0 || k == 3) ? 1 : -1, sy = (k < 2) ? 1 : -1;
        const double r2 = sqrt(2.0);
        const int mmax = min(p.nx, p.ny);
        for (int m = 0; m < mmax && n < cap; m++) {
            double lo = m == 0 ? 0.0 : r2 * (m - 0.5), hi = r2 * (m + 0.5);
            if (lo >= p.tb) break;
            lo = fmax(lo, p.ta);
            hi = fmin(hi, p.tb);
            if (hi > lo) emit(n++, m * sx, m * sy, hi - lo);
        }
        p.cnt[k] = n;
        return;
    }
    double wx, wy;
    sincospi(2.0 * ((double)k + 0.5) / (double)p.ndir, &wy, &wx);  // theta_k = 2 pi (k + 1/2)/N
    // no ray from a probe inside the box is still inside beyond tmax
    const double tmax = fmin((double)p.nx / fabs(wx), (double)p.ny / fabs(wy));
    const double ta = p.ta, tb = fmin(p.tb, tmax);
    if (!(ta < tb)) { p.cnt[k] = 0; return; }
    const double x0 = ta * wx, y0 = ta * wy;
    int ix = (int)floor(x0), iy = (int)floor(y0);
    if ((double)ix == x0 && wx < 0.0) ix--;
    if ((double)iy == y0 && wy < 0.0) iy--;
    const int sx = wx > 0.0 ? 1 : -1, sy = wy > 0.0 ? 1 : -1;
    int gx = wx > 0.0 ? ix + 1 : ix, gy = wy > 0.0 ? iy + 1 : iy;
    double tmx = (double)gx / wx, tmy = (double)gy / wy;  // irrational slopes: wx, wy never 0
    double t = ta;
    while (n < cap) {
        const double tn = fmin(fmin(tmx, tmy), tb);
        const double ds = tn - t;
        if (ds > 0.0) emit(n++, ix, iy, ds);
        if (tn >= tb) break;
        const bool stepx = tmx <= tmy, stepy = tmy <= tmx;
        if (stepx) { ix += sx; gx += sx; tmx = (double)gx / wx; }
        if (stepy) { iy += sy; gy += sy; tmy = (double)gy / wy; }
        t = tn;
    }
    p.cnt[k] = n;
}

cudaError_t launch_table_build(const TableBuildParams &p, cudaStream_t st) {
    const int threads = 128;
    const long long blocks = (p.ndir * (p.fix ? 16 : 1) + threads - 1) / threads;
    table_build_kernel<<<(unsigned)blocks, threads, 0, st>>>(p);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// March + merge.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2_neg(float tau2) {  // 2^-tau2, flushes to 0 below 2^-126
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(-tau2));
    return r;
}

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

template <int LV>
__device__ __forceinline__ void load_vec(const float *p, float (&v)[LV]) {
    if constexpr (LV == 8) {
        // one 256-bit load (sm_100: LDG.E.256): 32 B = one sector per lane
        asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
            : "l"(p));
    } else if constexpr (LV == 4) {
        const float4 a = __ldg(reinterpret_cast<const float4 *>(p));
        v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
    } else if constexpr (LV == 2) {
        const float2 a = __ldg(reinterpret_cast<const float2 *>(p));
        v[0] = a.x; v[1] = a.y;
    } else {
        v[0] = __ldg(p);
    }
}

// Predicated gather: lanes with pred == 0 issue no load and keep the (finite) values their registers
// already hold; the step length they integrate over is 0, so those values have no effect.
template <int LV>
__device__ __forceinline__ void load_vec_if(const float *p, float (&v)[LV], int pred) {
    if constexpr (LV == 8) {
        asm("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %9, 0;\n\t"
            "@q ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t}"
            : "+f"(v[0]), "+f"(v[1]), "+f"(v[2]), "+f"(v[3]), "+f"(v[4]), "+f"(v[5]), "+f"(v[6]), "+f"(v[7])
            : "l"(p), "r"(pred));
    } else if constexpr (LV == 4) {
        asm("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %5, 0;\n\t"
            "@q ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];\n\t}"
            : "+f"(v[0]), "+f"(v[1]), "+f"(v[2]), "+f"(v[3])
            : "l"(p), "r"(pred));
    } else if constexpr (LV == 2) {
        asm("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %3, 0;\n\t"
            "@q ld.global.nc.v2.f32 {%0,%1}, [%2];\n\t}"
            : "+f"(v[0]), "+f"(v[1])
            : "l"(p), "r"(pred));
    } else {
        asm("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %2, 0;\n\t"
            "@q ld.global.nc.f32 %0, [%1];\n\t}"
            : "+f"(v[0])
            : "l"(p), "r"(pred));
    }
}

template <int LV>
__device__ __forceinline__ void store_vec(float *p, const float (&v)[LV]) {
    if constexpr (LV == 8) {
        reinterpret_cast<float4 *>(p)[0] = make_float4(v[0], v[1], v[2], v[3]);
        reinterpret_cast<float4 *>(p)[1] = make_float4(v[4], v[5], v[6], v[7]);
    } else if constexpr (LV == 4) {
        reinterpret_cast<float4 *>(p)[0] = make_float4(v[0], v[1], v[2], v[3]);
    } else if constexpr (LV == 2) {
        reinterpret_cast<float2 *>(p)[0] = make_float2(v[0], v[1]);
    } else {
        p[0] = v[0];
    }
}

// ------------------------------------------------------------------------------------------------
// Pack: one thread per (batch, ym, xm, yd, xd); moves LV wavelengths of one cell.
// ------------------------------------------------------------------------------------------------
template <int LV>
__global__ void __launch_bounds__(256) pack_kernel(PackParams p) {
    const long long ncell = (long long)p.nx * p.ny;
    // thread -> (output cell c, batch nbI): 4 consecutive output cells x the batches are neighbours, so that a warp
    // reads whole cells (4 x nb LV floats: full 128-byte lines of the caller's arrays) and writes one full 128-byte
    // line per batch.  (Batch-slowest threads read one 32-byte sector of every cell at a time: 39 % of the HBM peak.)
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long grp = t >> 2;
    const int nbI = p.nb0 + (int)(grp % p.nb);          // (a launch covers batches nb0 .. nb0 + nb - 1)
    const long long c = (grp / p.nb) * 4 + (t & 3);  // output cell index ((ym*s + xm)*npy + yd)*npx + xd
    if (c >= ncell) return;
    // output order: batch-major planes for the lock-step and fan marches, cell records for the march over hit lists
    // (groups of list_b batches: [group][cell][batch in group][LV], the last group as wide as it is)
    long long idx = (long long)nbI * ncell + c;
    if (p.list_b > 0) {
        const int g0 = nbI / p.list_b * p.list_b, Bg = min(p.list_b, p.nb - g0);
        idx = (long long)g0 * ncell + c * Bg + (nbI - g0);
    }
    // small grids: one launch packs for every cascade (blockIdx.y), each into its own arrays
    const int shift = p.nmulti > 0 ? p.shifts[blockIdx.y] : p.shift;
    float *const chiT = p.nmulti > 0 ? p.chiTm[blockIdx.y] : p.chiT, *const ST = p.nmulti > 0 ? p.STm[blockIdx.y] : p.ST;
    const int npx = p.nx >> shift, npy = p.ny >> shift, smask = (1 << shift) - 1;
    const int xd = (int)(c % npx);
    long long r = c / npx;
    const int yd = (int)(r % npy);
    r /= npy;
    const int xm = (int)r & smask, ym = (int)(r >> shift);
    const int x = (xd << shift) + xm, y = (yd << shift) + ym;
    const long long src = ((long long)y * p.nx + x) * p.L + (long long)nbI * LV;
    float ch[LV], et[LV], c2[LV], S[LV];
    if ((nbI + 1) * LV <= p.L && (p.L % LV) == 0) {
        load_vec<LV>(p.chi + src, ch);  // one 32-byte sector per thread at LV = 8
        load_vec<LV>(p.eta + src, et);
    } else {
#pragma unroll
        for (int v = 0; v < LV; v++) {
            const bool ok = nbI * LV + v < p.L;
            ch[v] = ok ? __ldg(p.chi + src + v) : 0.f;
            et[v] = ok ? __ldg(p.eta + src + v) : 0.f;
        }
    }
#pragma unroll
    for (int v = 0; v < LV; v++) {
        // The march updates a channel in one of two forms (seg_update*()), and which one is decided HERE, per cell and
        // wavelength, from the opacity alone: optically thick enough (chi log2e >= c_thin) -> S = eta/chi, stored as it
        // is; thin -> -eta/2, the sign being the flag.  Emission without (or with next to no) opacity is thus valid
        // input and adds eta ds (eq. 16 in the limit chi -> 0, reading G11): the thin form never divides by chi.
        c2[v] = ch[v] * 1.4426950408889634f;             // tau in units of ln 2: T = 2^-tau2
        S[v] = c2[v] < p.c_thin ? (et[v] > 0.f ? -0.5f * et[v] : 0.f) : et[v] / ch[v];
    }
    if (p.active != nullptr && __ldg(p.active + (long long)y * p.nx + x) == 0) {
        // sparsity: "non-flagged cells are treated as transparent with no emission"
#pragma unroll
        for (int v = 0; v < LV; v++) { c2[v] = 0.f; S[v] = 0.f; }
    }
    float *oc = chiT + idx * LV, *os = ST + idx * LV;
    if constexpr (LV == 8) {
        reinterpret_cast<float4 *>(oc)[0] = make_float4(c2[0], c2[1], c2[2], c2[3]);
        reinterpret_cast<float4 *>(oc)[1] = make_float4(c2[4], c2[5], c2[6], c2[7]);
        reinterpret_cast<float4 *>(os)[0] = make_float4(S[0], S[1], S[2], S[3]);
        reinterpret_cast<float4 *>(os)[1] = make_float4(S[4], S[5], S[6], S[7]);
    } else if constexpr (LV == 4) {
        reinterpret_cast<float4 *>(oc)[0] = make_float4(c2[0], c2[1], c2[2], c2[3]);
        reinterpret_cast<float4 *>(os)[0] = make_float4(S[0], S[1], S[2], S[3]);
    } else if constexpr (LV == 2) {
        reinterpret_cast<float2 *>(oc)[0] = make_float2(c2[0], c2[1]);
        reinterpret_cast<float2 *>(os)[0] = make_float2(S[0], S[1]);
    } else {
        oc[0] = c2[0];
        os[0] = S[0];
    }
}

// Line mode: line [y][x][6] = chi_c, S_c, chi_line, S_line, v_x, v_y  ->  phase-plane layout, 6 floats per cell:
// chi_c log2e, chi_c log2e S_c, chi_line log2e/sqrt(pi), chi_line log2e/sqrt(pi) S_line, v_x sqrt(log2e), v_y sqrt(log2e)
// (tau in units of ln 2; phi(a) = 2^-(a sqrt(log2e))^2 / sqrt(pi)).
__global__ void __launch_bounds__(256) pack_line_kernel(PackParams p) {
    const long long ncell = (long long)p.nx * p.ny;
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const int npx = p.nx >> p.shift, npy = p.ny >> p.shift, smask = (1 << p.shift) - 1;
    const int xd = (int)(c % npx);
    long long t = c / npx;
    const int yd = (int)(t % npy);
    t /= npy;
    const int xm = (int)t & smask, ym = (int)(t >> p.shift);
    const int x = (xd << p.shift) + xm, y = (yd << p.shift) + ym;
    const float2 *src = reinterpret_cast<const float2 *>(p.chi + ((long long)y * p.nx + x) * 6);
    const float2 a = __ldg(src), b = __ldg(src + 1), v = __ldg(src + 2);
    const float L2E = 1.4426950408889634f, RSPI = 0.5641895835477563f, SL2E = 1.2011224087864498f;
    float cc = a.x * L2E, cl = b.x * L2E * RSPI;
    if (p.active != nullptr && __ldg(p.active + (long long)y * p.nx + x) == 0) { cc = 0.f; cl = 0.f; }  // not flagged: vacuum
    float2 *dst = reinterpret_cast<float2 *>(p.chiT + c * 6);
    dst[0] = make_float2(cc, cc * a.y);
    dst[1] = make_float2(cl, cl * b.y);
    dst[2] = make_float2(v.x * SL2E, v.y * SL2E);
}

cudaError_t launch_pack_line(const PackParams &p, cudaStream_t st) {
    const long long n = (long long)p.nx * p.ny;
    pack_line_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_pack(const PackParams &p, int LV, cudaStream_t st) {
    const long long n = (((long long)p.nx * p.ny + 3) / 4) * 4 * p.nb;
    const dim3 blocks((unsigned)((n + 255) / 256), (unsigned)(p.nmulti > 0 ? p.nmulti : 1));
    switch (LV) {
        case 8: pack_kernel<8><<<blocks, 256, 0, st>>>(p); break;
        case 4: pack_kernel<4><<<blocks, 256, 0, st>>>(p); break;
        case 2: pack_kernel<2><<<blocks, 256, 0, st>>>(p); break;
        default: pack_kernel<1><<<blocks, 256, 0, st>>>(p); break;
    }
    return cudaGetLastError();
}

// Streaming (evict-first) access for the banded launches' parked ray state: read once, written once.
template <int LV>
__device__ __forceinline__ void load_vec_cs(const float *p, float (&v)[LV]) {
    if constexpr (LV >= 4) {
#pragma unroll
        for (int q = 0; q < LV / 4; q++) {
            const float4 a = __ldcs(reinterpret_cast<const float4 *>(p) + q);
            v[4 * q] = a.x; v[4 * q + 1] = a.y; v[4 * q + 2] = a.z; v[4 * q + 3] = a.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < LV; q++) v[q] = __ldcs(p + q);
    }
}

template <int LV>
__device__ __forceinline__ void store_vec_cs(float *p, const float (&v)[LV]) {
    if constexpr (LV >= 4) {
#pragma unroll
        for (int q = 0; q < LV / 4; q++)
            __stcs(reinterpret_cast<float4 *>(p) + q, make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]));
    } else {
#pragma unroll
        for (int q = 0; q < LV; q++) __stcs(p + q, v[q]);
    }
}

// ------------------------------------------------------------------------------------------------
// eq. 16 for one cell, accurate at every optical depth.  x = chi ds log2 e is the optical depth of
// the segment in units of ln 2; tau accumulates (one rounding per cell) and T_n = 2^-tau_n.  The cell emits
// S T_(n-1) (1 - 2^-x), evaluated in one of two forms chosen per cell and channel by pack_kernel (from chi alone, so
// that the march spends no multiplication on the decision; the sign of the packed source term is the flag):
//   thick (chi log2e >= c_thin = 1/64 / max over inclinations of 1/sin):  S (T_(n-1) - T_n), S = eta/chi packed.
//       Difference of two transmittances, each good to ~1e-7 T: relative error < 2e-5 per cell of typical length, and
//       the roundings of T_n cancel between neighbouring cells
//   thin:  (eta/2) ds (T_(n-1) + T_n), -eta/2 packed.  Trapezoid of the attenuation across the cell:
//       1 - e^-y = (y/2)(1 + e^-y)(1 - y^2/12 + ...), y = x ln 2 <= 0.0153: relative error < 2e-5; exact as chi -> 0
//       (eta ds T, reading G11) and blind to the resolution of T, so optically thin rays and thin emitters behind
//       absorbers keep their emission
// One form for every launch: there is no "thin" kernel variant and no host-side detection.
// Channels are processed two at a time with the packed fp32 instructions of sm_100 (FFMA2 / FADD2 / FMUL2).
// ------------------------------------------------------------------------------------------------
static constexpr float KAPPA = 0.34657359027997264f;  // ln 2 / 2   (line mode, where chi is evaluated per ray)
static constexpr float XK_THIN = KAPPA / 64.f;         // line mode: threshold on x ln2 / 2

typedef unsigned long long f32x2;  // two floats in one 64-bit register pair (lo, hi)
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void up2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

// two channels: c = chi log2e, S = packed source term (eta/chi, or -eta/2 in a thin cell), ds = path length, mds = -ds
// (pairs); state tau, T, I (pairs)
__device__ __forceinline__ void seg_update2(f32x2 c, f32x2 S, f32x2 ds, f32x2 mds, f32x2 &tau, f32x2 &T, f32x2 &I) {
    tau = fma2(c, ds, tau);
    float t0, t1;
    up2(tau, t0, t1);
    const f32x2 Tn = pk2(ex2_neg(t0), ex2_neg(t1));
    const f32x2 d = sub2(T, Tn), ms = mul2(add2(T, Tn), mds);
    float s0, s1, d0, d1, m0, m1;
    up2(S, s0, s1);
    up2(d, d0, d1);
    up2(ms, m0, m1);
    I = fma2(S, pk2(s0 < 0.f ? m0 : d0, s1 < 0.f ? m1 : d1), I);
    T = Tn;
}

// one channel (single-wavelength launches)
__device__ __forceinline__ void seg_update1(float c, float S, float ds, float &tau, float &T, float &I) {
    tau = fmaf(c, ds, tau);
    const float Tn = ex2_neg(tau);
    I = fmaf(S, S < 0.f ? -ds * (T + Tn) : T - Tn, I);
    T = Tn;
}

// line mode, two channels: a = x_l + v.w (pairs), the six packed line parameters of the cell broadcast; profile, opacity,
// emissivity and the update of seg_update2 with S = num / chi (thin branch: num dk (T + Tn), no division involved)
__device__ __forceinline__ void seg_update_line2(f32x2 aa, float cc, float ccS, float cl, float clS, f32x2 ds, f32x2 dk, f32x2 &tau, f32x2 &T, f32x2 &I) {
    float q0, q1;
    up2(mul2(aa, aa), q0, q1);
    const f32x2 phi = pk2(ex2_neg(q0), ex2_neg(q1));
    const f32x2 c = fma2(pk2(cl, cl), phi, pk2(cc, cc)), num = fma2(pk2(clS, clS), phi, pk2(ccS, ccS));
    float c0, c1;
    up2(c, c0, c1);
    // pack_line_kernel keeps chi_c >= 1e-37 where the cell holds anything, so c > 0 there; exact vacuum: num = 0, guarded
    const f32x2 Sv = mul2(num, pk2(c0 > 0.f ? rcp_approx(c0) : 0.f, c1 > 0.f ? rcp_approx(c1) : 0.f));
    tau = fma2(c, ds, tau);
    const f32x2 xk = mul2(c, dk);
    float t0, t1;
    up2(tau, t0, t1);
    const f32x2 Tn = pk2(ex2_neg(t0), ex2_neg(t1));
    const f32x2 thick = mul2(Sv, sub2(T, Tn)), thin = mul2(mul2(num, dk), add2(T, Tn));
    float x0, x1, a0, a1, b0, b1;
    up2(xk, x0, x1);
    up2(thick, a0, a1);
    up2(thin, b0, b1);
    I = add2(I, pk2(x0 < XK_THIN ? b0 : a0, x1 < XK_THIN ? b1 : a1));
    T = Tn;
}

// line mode: the cell's eta log2e (num) and chi log2e (c) are evaluated per ray; emission eta ds T in the thin branch
__device__ __forceinline__ void seg_update_line(float c, float num, float ds, float dk, float &tau, float &T, float &I) {
    const float Sv = c > 0.f ? __fdividef(num, c) : 0.f;  // eta/chi
    tau = fmaf(c, ds, tau);
    const float xk = c * dk, Tn = ex2_neg(tau);
    I += xk < XK_THIN ? (num * dk) * (T + Tn) : Sv * (T - Tn);
    T = Tn;
}

// Position of child probe a among the n parents per axis: a/2 - 1/4 in parent index units, clamped
// at the lattice edge.  Weight `f` goes to q1.
__device__ __forceinline__ void parent_axis(int a, int n, int &q0, int &q1, float &f) {
    const int base = (a & 1) ? (a - 1) >> 1 : (a >> 1) - 1;
    f = (a & 1) ? 0.25f : 0.75f;
    q0 = min(max(base, 0), n - 1);
    q1 = min(max(base + 1, 0), n - 1);
}

// Warp -> work mapping shared by march_kernel and count_kernel.  One warp = one PATCH of pw x ph = 32
// probes (lanes) x one direction group.  Warps are numbered flat: the G = min(ngroups, 8) adjacent
// direction groups of one patch are neighbours (their rays overlap near the probes), then the patch,
// then the remaining direction bits, then the wavelength batch: the warps resident at any time
// share a narrow fan of directions (a few MB of step tables) and one batch's planes (L2).
struct WarpWork {
    int nbI, kg, a, b;
    int cls;        // bilinear fix: parity class (a & 1) + 2 (b & 1) of the warp's probes
    unsigned gidx;  // the lane's own entry in a phase plane of the packed layout (gather base)
    bool any, valid;
};

__device__ __forceinline__ WarpWork warp_work(const MarchParams &p, long long W, int lane) {
    if (p.cpw) W >>= 2;  // child-per-warp: 4 consecutive warps (one per child direction) share everything else
    const int G = min(p.kg_n, 8);
    const int ncls = p.fix ? 4 : 1;
    const long long npatch = p.qlist != nullptr ? (long long)(p.qpad >> 3) * ncls : p.plist != nullptr ? p.npatch_act : (long long)p.npatch_x * p.npatch_y * ncls;
    WarpWork r;
    const int kg_lo = (int)(W % G);
    W /= G;
    long long patch = W % npatch;
    W /= npatch;
    if (p.qlist != nullptr) {
        // sorted quads (unbanded dense launches without the fix): lanes 4q .. 4q+3 are the probes of the q-th quad of this
        // warp's 8 entries of the list of its block of direction groups
        const int kgb_n = p.kg_n / G, kgb = (int)(W % kgb_n);
        r.kg = (kgb * G + kg_lo + p.kg_off) & (p.ngroups - 1);
        r.nbI = (int)(W / kgb_n);
        r.any = r.nbI < p.nb;
        r.nbI += p.nb0;
        // (bilinear fix: the lattice of one parity class, spacing 2s; the same list serves the four classes)
        r.cls = (int)(patch % ncls);
        patch /= ncls;
        const unsigned q = __ldg(p.qlist + (long long)kgb * p.qpad + patch * 8 + (lane >> 2));
        const int lxq = p.fix ? p.npx >> 1 : p.npx, qx = lxq >> 2;
        r.valid = q != 0xffffu;
        const int lbq = r.valid ? (int)(q / qx) : 0, laq = r.valid ? (int)(q - (unsigned)lbq * qx) * 4 + (lane & 3) : 0;
        r.a = p.fix ? 2 * laq + (r.cls & 1) : laq;
        r.b = p.fix ? 2 * lbq + (r.cls >> 1) : lbq;
        r.gidx = (unsigned)lbq * lxq + laq;
        return r;
    }
    // sparsity: only the patches that hold a flagged probe are launched (plist: their numbers, in order)
    if (p.plist != nullptr) patch = __ldg(p.plist + patch);
    r.cls = (int)(patch % ncls);
    patch /= ncls;
    const int kgb_n = p.kg_n / G;
    // a launch covers kg_n consecutive direction groups starting at kg_off, modulo the full circle
    r.kg = ((int)(W % kgb_n) * G + kg_lo + p.kg_off) & (p.ngroups - 1);
    r.nbI = (int)(W / kgb_n);
    r.any = r.nbI < p.nb;
    r.nbI += p.nb0;  // (a launch covers batches nb0 .. nb0 + nb - 1)
    const int py = (int)(patch / p.npatch_x), px = (int)(patch - (long long)py * p.npatch_x);
    const int pw = 1 << p.pw_log2;
    // lane lattice: all probes, or (bilinear fix) the probes of one parity class, spacing 2s
    const int la = (px << p.pw_log2) + (lane & (pw - 1)), lb = py * (32 >> p.pw_log2) + (lane >> p.pw_log2);
    const int lx = p.fix ? p.npx >> 1 : p.npx, ly = p.fix ? p.npy >> 1 : p.npy;
    r.valid = la < lx && lb < ly;
    r.a = p.fix ? 2 * la + (r.cls & 1) : la;
    r.b = p.fix ? 2 * lb + (r.cls >> 1) : lb;
    r.gidx = (unsigned)lb * lx + la;
    // a probe that is not flagged computes nothing and writes nothing; nothing flagged ever reads it
    if (r.valid && p.flags != nullptr) r.valid = __ldg(p.flags + (long long)r.b * p.npx + r.a) != 0;
    if (!r.valid) { r.a = r.cls & 1; r.b = r.cls >> 1; r.gidx = 0; }
    return r;
}

__host__ __device__ inline long long march_warps(const MarchParams &p) {
    const long long npatch = p.qlist != nullptr ? (long long)(p.qpad >> 3) * (p.fix ? 4 : 1) : p.plist != nullptr ? p.npatch_act : (long long)p.npatch_x * p.npatch_y * (p.fix ? 4 : 1);
    return npatch * p.kg_n * p.nb * (p.cpw ? 4 : 1);
}

// Number of leading steps of direction k's table that lie inside the box for this lane's probe.
// The box is convex and the probe is inside it, so the in-box steps are a prefix; dx and dy are
// monotone along the ray, so the first step outside is found by bisection on the (dx, dy) table.
__device__ __forceinline__ int steps_inside(const StepXY *xy, int n, bool valid, int dxlo, int dxhi, int dylo, int dyhi) {
    int lo = 0, hi = valid ? n : 0;  // smallest st in [0, n] that is outside (n: none is)
    const int iters = 32 - __clz(n);  // ceil(log2(n + 1)); warp-uniform
    for (int it = 0; it < iters; it++) {
        const int mid = (lo + hi) >> 1;
        if (lo < hi) {
            const unsigned e = __ldg(reinterpret_cast<const unsigned *>(xy) + mid);
            const int dx = (int)(short)(e & 0xffffu), dy = (int)(short)(e >> 16);
            const bool out = dx < dxlo || dx > dxhi || dy < dylo || dy > dyhi;
            if (out) hi = mid; else lo = mid + 1;
        }
    }
    return lo;
}

// Banded launches (grids whose wavelength batch does not fit L2): first step st in [0, n] whose cell
// coordinate along the band axis, c0 + d(st), has reached `thr` in the ray's direction of travel
// (sg = +1: c >= thr, sg = -1: c <= thr).  d is monotone along the ray, so this is a bisection.
__device__ __forceinline__ int first_step_reaching(const StepXY *xy, int n, int axis, int sg, int c0, int thr) {
    int lo = 0, hi = n;
    const int iters = 32 - __clz(n);
    for (int it = 0; it < iters; it++) {
        const int mid = (lo + hi) >> 1;
        if (lo < hi) {
            const unsigned e = __ldg(reinterpret_cast<const unsigned *>(xy) + mid);
            const int d = axis ? (int)(short)(e & 0xffffu) : (int)(short)(e >> 16);
            const bool reached = sg * (c0 + d) >= sg * thr;
            if (reached) hi = mid; else lo = mid + 1;
        }
    }
    return lo;
}

// One warp = 32 probes (a pw x ph patch of the probe lattice) x 1 direction group (its 4 child
// directions in turn) x LV wavelengths per lane.  Per step the warp reads one 8-byte table entry
// (uniform address) and each lane its cell's LV opacities and source functions.  The gathers run
// PD steps ahead of the integration in a register ring (slot = step mod PD, loop unrolled by PD):
// while step st is integrated the loads of steps st+1 .. st+PD-1 are in flight.
//
// BANDED: the launch covers only the steps inside one band of rows (or columns) of the grid and only the
// half of the directions that crosses the bands in ascending (or descending) order; a ray's (I, tau)
// is carried from band to band through `state`, so the arithmetic - and the result - is that of the
// unbanded launch, bit for bit, while the cells gathered by one launch fit L2.
template <int LV, int NM, int PD, int WARPS, int MINB, bool BANDED, bool LINE>
__global__ void __launch_bounds__(WARPS * 32, MINB) march_kernel(MarchParams p) {
    // sum over the 4 child directions, per thread: parked in shared memory between children so the
    // marching loop has the registers to itself
    constexpr int LL = LV / NM;  // wavelengths per lane; channel ch = l * NM + m (inclination fastest)
    __shared__ float acc_s[LV][WARPS * 32];
    const int lane = threadIdx.x & 31;
    const long long W = (long long)blockIdx.x * WARPS + (threadIdx.x >> 5);
    const WarpWork ww = warp_work(p, W, lane);
    if (!ww.any) return;
    const int nbI = ww.nbI, kg = ww.kg, a = ww.a, b = ww.b;
    const bool valid = ww.valid;
    const unsigned probe = (unsigned)b * p.npx + a;  // output / parked-state index
    const unsigned gidx = ww.gidx;                    // gather base in the packed layout
    const int half = (1 << p.shift) >> 1;
    const int Y0 = (b << p.shift) + half;
    const long long ncell = (long long)p.nx * p.ny;
    // packed layout [batch][y mod s][x mod s][y div s][x div s][LV]: the lane's probe owns cell
    // (y div s, x div s) = (b, a) of every phase plane; a step's delta is lane-independent
    const float *chiB = LINE ? p.linepk : p.chiT + (long long)nbI * ncell * LL;  // warp-uniform
    const float *SB = LINE ? nullptr : p.ST + (long long)nbI * ncell * LL;
    // LINE: the packed cell holds the 6 line parameters; chi and S of each wavelength are
    // evaluated per step from the velocity projected on this ray.  xs = x_l sqrt(log2 e) of the lane's wavelengths.
    constexpr int NR = LINE ? 6 : LL;  // floats gathered per cell
    float xs[LINE ? LL : 1];
    if constexpr (LINE) {
#pragma unroll
        for (int v = 0; v < LL; v++) xs[v] = __ldg(p.xls + nbI * LL + v);
    }
    // (dx, dy) ranges that keep this lane's ray inside the box
    const int dxlo = -(a << p.shift) - half, dxhi = ((p.npx - a) << p.shift) - 1 - half;
    const int dylo = -Y0, dyhi = p.ny - 1 - Y0;

#pragma unroll
    for (int v = 0; v < LV; v++) acc_s[v][threadIdx.x] = 0.f;

    // bilinear fix (p.fix): every ray is traced four times, once towards each parent (slot)
    const int nsub = p.fix ? 4 : 1;
    // child-per-warp (p.cpw): the 4 child directions of a group run in 4 neighbouring warps at the same time, so
    // that the cells two adjacent directions share (13-16 % of them) are found in L1; the 4 partial results meet in
    // shared memory and are summed in the same order as by a single warp.  The warps start together and their rays
    // are equally long, so they stay close on their own: named barriers every few steps were measured and cost
    // more than the extra hits bring (76.2 against 73.6 ms on config 2).
    const int jj0 = p.cpw ? (int)(W & 3) * nsub : 0, jj1 = p.cpw ? jj0 + nsub : 4 * nsub;
    for (int jj = jj0; jj < jj1; jj++) {
        const int j = p.fix ? jj >> 2 : jj, slot = p.fix ? jj & 3 : 0;
        const long long k = 4LL * kg + j;
        const long long tid = p.fix ? k * 16 + ww.cls * 4 + slot : k;  // table of this (sub-)ray
        float I[LV], tau[LV], T[LV];
#pragma unroll
        for (int v = 0; v < LV; v++) { I[v] = 0.f; tau[v] = 0.f; T[v] = 1.f; }
        // cnt == null: the whole cascade lies outside any box of this size (pure boundary term)
        if (p.cnt != nullptr) {
            const long long o = __ldg(p.off + tid);
            const int n = __ldg(p.cnt + tid);
            const uint2 *tab = reinterpret_cast<const uint2 *>(p.steps + o);
            int nin = steps_inside(p.xy + o, n, valid, dxlo, dxhi, dylo, dyhi);
            if (p.fix && n > 0) {  // a sub-ray that starts outside the box is vacuum (reading G10)
                const unsigned e = __ldg(reinterpret_cast<const unsigned *>(p.xy + o));
                const int dx = (int)(short)(e & 0xffffu), dy = (int)(short)(e >> 16);
                if (dx < dxlo || dx > dxhi || dy < dylo || dy > dyhi) nin = 0;
            }
            bool has = true;  // banded: the lane has steps in this band
            int n0 = 0;       // this lane's first step of this launch
            if constexpr (BANDED) {
                const int c0 = p.band_axis ? (a << p.shift) + half : Y0;
                const int sg = p.band_sign;
                // steps [n0, n1) of this launch: those inside rows/columns [band_lo, band_hi)
                n0 = min(nin, first_step_reaching(p.xy + o, n, p.band_axis, sg, c0, sg > 0 ? p.band_lo : p.band_hi - 1));
                const int n1 = min(nin, first_step_reaching(p.xy + o, n, p.band_axis, sg, c0, sg > 0 ? p.band_hi : p.band_lo - 1));
                has = n1 > n0;
                if (valid && n0 > 0 && (has || p.band_final)) {  // steps were taken in earlier bands: resume
                    const float *stp = p.state + ((((long long)nbI * p.ngroups + kg) * 4 + j) * ((long long)p.npx * p.npy) + probe) * (2 * LV);
                    load_vec_cs<LV>(stp, I);
                    load_vec_cs<LV>(stp + LV, tau);
#pragma unroll
                    for (int v = 0; v < LV; v++) T[v] = ex2_neg(tau[v]);
                }
                int w0 = __reduce_min_sync(FULL, has ? n0 : 0x7fffffff);  // the warp's first step
                if (w0 == 0x7fffffff) w0 = 0;
                tab += w0;  // from here on step indices are relative to the warp's first step
                nin = has ? n1 - w0 : 0;
                n0 = has ? n0 - w0 : 0;
            }
            const int nw = __reduce_max_sync(FULL, nin);  // steps this warp walks
            float c2[PD][NR], S[PD][LINE ? 1 : LL], ds[PD];
            // LINE: photons on this ray travel along -(wx, wy); the line of a cell moving with v is centred at
            // x = -v.w, so a = x_l + v.w  (packed v and x_l carry the factor sqrt(log2 e): phi ~ 2^(-a^2))
            float wx = 0.f, wy = 0.f;
            if constexpr (LINE) {
                if (p.fix) { const float2 d = __ldg(p.subdir + tid); wx = d.x; wy = d.y; }
                else sincospif(2.f * ((float)k + 0.5f) / (float)(4LL * p.ngroups), &wy, &wx);
            }
            auto gather = [&](int u, unsigned delta, bool in) {
                if constexpr (LINE) {
                    const float *src = reinterpret_cast<const float *>(reinterpret_cast<const char *>(chiB) +
                                                                        (unsigned long long)(gidx + delta) * 24ull);
                    float t0[2] = {c2[u][0], c2[u][1]}, t1[2] = {c2[u][2], c2[u][3]}, t2[2] = {c2[u][4], c2[u][5]};
                    load_vec_if<2>(src, t0, in);
                    load_vec_if<2>(src + 2, t1, in);
                    load_vec_if<2>(src + 4, t2, in);
                    c2[u][0] = t0[0]; c2[u][1] = t0[1]; c2[u][2] = t1[0]; c2[u][3] = t1[1]; c2[u][4] = t2[0]; c2[u][5] = t2[1];
                } else {
                    const unsigned long long d = (unsigned long long)(gidx + delta) * (LL * sizeof(float));
                    load_vec_if<LL>(reinterpret_cast<const float *>(reinterpret_cast<const char *>(chiB) + d), c2[u], in);
                    load_vec_if<LL>(reinterpret_cast<const float *>(reinterpret_cast<const char *>(SB) + d), S[u], in);
                }
            };
            // prologue: steps 0 .. PD-1 into the ring (the table has 2 PD spare entries at its end)
#pragma unroll
            for (int u = 0; u < PD; u++) {
#pragma unroll
                for (int v = 0; v < NR; v++) c2[u][v] = 0.f;
#pragma unroll
                for (int v = 0; v < (LINE ? 1 : LL); v++) S[u][v] = 0.f;
                const uint2 e = __ldg(tab + u);
                const bool in = u < nin && (!BANDED || u >= n0);
                gather(u, e.x, in);
                ds[u] = in ? __uint_as_float(e.y) : 0.f;
            }
            int chk = 0;
            // the channels of a lane two at a time (FFMA2 / FADD2 / FMUL2).  Pair q holds, when the lane has at least two
            // wavelengths, inclination q % NM of wavelengths 2 (q / NM) and 2 (q / NM) + 1 (two neighbouring gathered values,
            // one path length); with a single wavelength, inclinations 2q and 2q + 1 of it (one gathered value, two lengths)
            constexpr bool PACKED = LV >= 2;
            constexpr int NP = PACKED ? LV / 2 : 1;
            [[maybe_unused]] f32x2 I2[NP], tau2[NP], T2[NP];
            [[maybe_unused]] auto ch_lo = [](int q) { return LL >= 2 ? (2 * (q / NM)) * NM + q % NM : 2 * q; };
            [[maybe_unused]] auto ch_hi = [](int q) { return LL >= 2 ? (2 * (q / NM) + 1) * NM + q % NM : 2 * q + 1; };
            if constexpr (PACKED) {
#pragma unroll
                for (int q = 0; q < NP; q++) {
                    I2[q] = pk2(I[ch_lo(q)], I[ch_hi(q)]);
                    tau2[q] = pk2(tau[ch_lo(q)], tau[ch_hi(q)]);
                    T2[q] = pk2(T[ch_lo(q)], T[ch_hi(q)]);
                }
            }
            // a1: eq. 16 along the interval, front to back, seg_update*() per cell and channel
            int st_done = nw;  // steps the warp took (early exit: fewer)
            for (int st = 0; st < nw; st += PD) {
#pragma unroll
                for (int u = 0; u < PD; u++) {
                    const uint2 en = __ldg(tab + st + u + PD);
                    // integrate step st + u (a slot past the lane's last in-box step has ds = 0: no effect)
                    // 2.5D: inclination m crosses the same cell over ds / sin(inclination)
                    float dsm[NM], dkm[NM];  // dkm: ds ln2/2 in line mode, -ds otherwise (thin form of seg_update*())
#pragma unroll
                    for (int m = 0; m < NM; m++) {
                        dsm[m] = NM == 1 ? ds[u] : ds[u] * p.incl_f[m];
                        dkm[m] = LINE ? dsm[m] * KAPPA : -dsm[m];
                    }
                    if constexpr (LINE) {
                        // packed cell: chi_c', chi_c' S_c, chi_line', chi_line' S_line, v_x', v_y'   (' = scaled, pack_line_kernel)
                        // inclination m sees the in-plane velocity projected with sin(inclination) (2.5D line mode)
                        const float vw = fmaf(c2[u][4], wx, c2[u][5] * wy);
                        float vwm[NM];
#pragma unroll
                        for (int m = 0; m < NM; m++) vwm[m] = NM == 1 ? vw : vw * p.incl_s[m];
                        if constexpr (PACKED) {
#pragma unroll
                            for (int q = 0; q < NP; q++) {
                                if constexpr (LL >= 2) {
                                    const int l = 2 * (q / NM), m = q % NM;
                                    seg_update_line2(add2(pk2(xs[l], xs[l + 1]), pk2(vwm[m], vwm[m])), c2[u][0], c2[u][1], c2[u][2], c2[u][3],
                                                     pk2(dsm[m], dsm[m]), pk2(dkm[m], dkm[m]), tau2[q], T2[q], I2[q]);
                                } else {
                                    seg_update_line2(add2(pk2(xs[0], xs[0]), pk2(vwm[2 * q], vwm[2 * q + 1])), c2[u][0], c2[u][1], c2[u][2], c2[u][3],
                                                     pk2(dsm[2 * q], dsm[2 * q + 1]), pk2(dkm[2 * q], dkm[2 * q + 1]), tau2[q], T2[q], I2[q]);
                                }
                            }
                        } else {
#pragma unroll
                            for (int v = 0; v < LV; v++) {
                                const float aa = xs[v / NM] + vwm[v % NM];
                                const float phi = ex2_neg(aa * aa);
                                const float chi2 = fmaf(c2[u][2], phi, c2[u][0]);
                                const float num = fmaf(c2[u][3], phi, c2[u][1]);
                                seg_update_line(chi2, num, dsm[v % NM], dkm[v % NM], tau[v], T[v], I[v]);
                            }
                        }
                    } else {
                        if constexpr (PACKED) {
#pragma unroll
                            for (int q = 0; q < NP; q++) {
                                if constexpr (LL >= 2) {
                                    const int l = 2 * (q / NM), m = q % NM;
                                    seg_update2(pk2(c2[u][l], c2[u][l + 1]), pk2(S[u][l], S[u][l + 1]), pk2(dsm[m], dsm[m]),
                                                pk2(dkm[m], dkm[m]), tau2[q], T2[q], I2[q]);
                                } else {
                                    seg_update2(pk2(c2[u][0], c2[u][0]), pk2(S[u][0], S[u][0]), pk2(dsm[2 * q], dsm[2 * q + 1]),
                                                pk2(dkm[2 * q], dkm[2 * q + 1]), tau2[q], T2[q], I2[q]);
                                }
                            }
                        } else {
#pragma unroll
                            for (int v = 0; v < LV; v++)
                                seg_update1(c2[u][v / NM], S[u][v / NM], dsm[v % NM], tau[v], T[v], I[v]);
                        }
                    }
                    // refill the slot with step st + u + PD
                    const bool in = st + u + PD < nin && (!BANDED || st + u + PD >= n0);
                    gather(u, en.x, in);
                    ds[u] = in ? __uint_as_float(en.y) : 0.f;
                }
                if (p.early_exit && (++chk & 3) == 0) {
                    if constexpr (PACKED) {
#pragma unroll
                        for (int q = 0; q < NP; q++) up2(tau2[q], tau[ch_lo(q)], tau[ch_hi(q)]);
                    }
                    float tmin = tau[0];
#pragma unroll
                    for (int v = 1; v < LV; v++) tmin = fminf(tmin, tau[v]);
                    // every live lane opaque at every wavelength: T is exactly 0, nothing more can arrive
                    if (__all_sync(FULL, st + PD >= nin || tmin > p.tau_cut)) { st_done = st + PD; break; }
                }
            }
            if (p.walked != nullptr) {  // measurement only (rc_count_walked): in-box steps this launch integrated
                unsigned long long mine = (unsigned long long)max(0, min(nin, st_done) - n0);
                for (int sh = 16; sh > 0; sh >>= 1) mine += __shfl_down_sync(FULL, mine, sh);
                if (lane == 0 && mine) atomicAdd(p.walked, mine);
            }
            if constexpr (PACKED) {
#pragma unroll
                for (int q = 0; q < NP; q++) {
                    up2(I2[q], I[ch_lo(q)], I[ch_hi(q)]);
                    up2(tau2[q], tau[ch_lo(q)], tau[ch_hi(q)]);
                    up2(T2[q], T[ch_lo(q)], T[ch_hi(q)]);
                }
            }
            if constexpr (BANDED) {
                if (!p.band_final) {  // park the ray; the launch of its next band resumes it
                    if (valid && has) {
                        float *stp = p.state + ((((long long)nbI * p.ngroups + kg) * 4 + j) * ((long long)p.npx * p.npy) + probe) * (2 * LV);
                        store_vec_cs<LV>(stp, I);
                        store_vec_cs<LV>(stp + LV, tau);
                    }
                    continue;
                }
            }
        }
        const long long ndir = 4LL * p.ngroups;
        if (p.Aup == nullptr) {
            // a2: boundary intensity enters on the top cascade only: rays heading up
            // (sin theta_k > 0  <=>  k < N/2) see I_above, rays heading down I_below
            const float *Ib = (2 * k < ndir) ? p.I_above : p.I_below;
#pragma unroll
            for (int v = 0; v < LV; v++) I[v] = fmaf(T[v], __ldg(Ib + nbI * LV + v), I[v]);  // [wavelength][inclination]
        } else if (valid && p.fix) {
            // a3 with the bilinear fix: this sub-ray ends where parent `slot`'s child cone starts; merge it with that
            // parent alone (eq. 11), then weight it bilinearly.  At the lattice edge both slots of an axis are the
            // same (clamped) parent, reached by the ray of the slot that is NOT clamped: that slot takes the whole
            // weight (the oracle traces the same ray twice, with weights 1/4 + 3/4).
            const int npxu = p.npx >> 1, npyu = p.npy >> 1;
            int a0, a1, b0, b1;
            float fa, fb;
            parent_axis(a, npxu, a0, a1, fa);
            parent_axis(b, npyu, b0, b1, fb);
            const int sa = slot & 1, sb = slot >> 1;
            const int base_a = (a & 1) ? (a - 1) >> 1 : (a >> 1) - 1, base_b = (b & 1) ? (b - 1) >> 1 : (b >> 1) - 1;
            float wa = sa ? fa : 1.f - fa, wb = sb ? fb : 1.f - fb;
            if (base_a < 0) wa = sa ? 1.f : 0.f;
            if (base_a + 1 > npxu - 1) wa = sa ? 0.f : 1.f;
            if (base_b < 0) wb = sb ? 1.f : 0.f;
            if (base_b + 1 > npyu - 1) wb = sb ? 0.f : 1.f;
            const float *up = p.Aup + (((long long)nbI * ndir + k) * npyu) * (long long)npxu * LV;
            float uq[LV];
            load_vec<LV>(up + ((long long)(sb ? b1 : b0) * npxu + (sa ? a1 : a0)) * LV, uq);
            const float wq = wa * wb;
#pragma unroll
            for (int v = 0; v < LV; v++) I[v] = wq * fmaf(T[v], uq[v], I[v]);
        } else if (valid) {
            // a3: bilinear over the 4 parents of cascade i+1 (already averaged over the 4 children of
            // direction k when they were written), then eq. 11: I <- I + T * U
            const int npxu = p.npx >> 1, npyu = p.npy >> 1;
            int a0, a1, b0, b1;
            float fa, fb;
            parent_axis(a, npxu, a0, a1, fa);
            parent_axis(b, npyu, b0, b1, fb);
            const float *up = p.Aup + (((long long)nbI * ndir + k) * npyu) * (long long)npxu * LV;
            float u00[LV], u01[LV], u10[LV], u11[LV];
            load_vec<LV>(up + ((long long)b0 * npxu + a0) * LV, u00);
            load_vec<LV>(up + ((long long)b0 * npxu + a1) * LV, u01);
            load_vec<LV>(up + ((long long)b1 * npxu + a0) * LV, u10);
            load_vec<LV>(up + ((long long)b1 * npxu + a1) * LV, u11);
#pragma unroll
            for (int v = 0; v < LV; v++) {
                const float lo = fmaf(fa, u01[v] - u00[v], u00[v]);
                const float hi = fmaf(fa, u11[v] - u10[v], u10[v]);
                I[v] = fmaf(T[v], fmaf(fb, hi - lo, lo), I[v]);
            }
        }
#pragma unroll
        for (int v = 0; v < LV; v++) acc_s[v][threadIdx.x] += I[v];
    }
    if (p.cpw) {
        // the 4 warps of the group: named barrier, then the first of them adds the others' sums in child order
        const int g = (threadIdx.x >> 7);
        asm volatile("bar.sync %0, 128;" ::"r"(g + 1) : "memory");
        if ((W & 3) != 0) return;
#pragma unroll
        for (int v = 0; v < LV; v++)
            acc_s[v][threadIdx.x] = ((acc_s[v][threadIdx.x] + acc_s[v][threadIdx.x + 32]) + acc_s[v][threadIdx.x + 64]) + acc_s[v][threadIdx.x + 96];
    }
    if (!valid) return;
    if constexpr (BANDED) {
        if (!p.band_final) return;
    }
    const long long nprobe = (long long)p.npx * p.npy;
    float acc[LV];
#pragma unroll
    for (int v = 0; v < LV; v++) acc[v] = 0.25f * acc_s[v][threadIdx.x];  // mean over the 4 children (cascade 0: a4, J)
    if (p.mode == 0) {
        store_vec<LV>(p.out + (((long long)nbI * p.ngroups + kg) * nprobe + probe) * LV, acc);
        return;
    }
    // cascade 0: J_l = sum over the inclinations of w_m x (mean of the 4 directions)  (a4)
    float Jl[LL];
#pragma unroll
    for (int l = 0; l < LL; l++) {
        Jl[l] = NM == 1 ? acc[l] : 0.f;
        if constexpr (NM > 1) {
#pragma unroll
            for (int m = 0; m < NM; m++) Jl[l] = fmaf(p.incl_w[m], acc[l * NM + m], Jl[l]);
        }
    }
    if (p.mode == 1) {
        float *o = p.out + (long long)probe * p.L + nbI * LL;
        if ((nbI + 1) * LL <= p.L && (p.L % LL) == 0) {
            store_vec<LL>(o, Jl);
        } else {
#pragma unroll
            for (int v = 0; v < LL; v++)
                if (nbI * LL + v < p.L) o[v] = Jl[v];
        }
    } else {
        float sum = 0.f;
#pragma unroll
        for (int v = 0; v < LL; v++) sum = fmaf(__ldg(p.weights + nbI * LL + v), Jl[v], sum);
        p.out[(long long)nbI * nprobe + probe] = sum;
    }
}

template <int LV, int NM, int PD, int WARPS, int MINB>
static cudaError_t launch_march_variant(const MarchParams &p, cudaStream_t st) {
    const long long blocks = (march_warps(p) + WARPS - 1) / WARPS;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (blocks == 0) return cudaSuccess;  // sparsity: no flagged probe in this cascade
    if (p.state != nullptr)
        march_kernel<LV, NM, PD, WARPS, MINB, true, false><<<(unsigned)blocks, WARPS * 32, 0, st>>>(p);
    else
        march_kernel<LV, NM, PD, WARPS, MINB, false, false><<<(unsigned)blocks, WARPS * 32, 0, st>>>(p);
    return cudaGetLastError();
}

// variant: 0 = ring of 2 steps, 24 warps/SM (<= 80 registers); 1 = ring of 3, 20 warps/SM (<= 96, blocks of 4 warps);
//          2 = ring of 3, 16 warps/SM (<= 128); 3 = ring of 4, 16 warps/SM (<= 128); 4 = ring of 2, 20 warps/SM (<= 96)
// ------------------------------------------------------------------------------------------------
// Mostly empty atmospheres ("accelerating the traversal of long-range radiance intervals through
// free-space"): the FAN march.  The packed arrays are in plain cell order (shift 0) and every lane walks its OWN ray: it
// looks its cell up in `dist` - the Chebyshev distance to the nearest occupied cell, 0 = occupied - and jumps over the
// steps that cannot meet one; only occupied cells are gathered and integrated.  An empty cell changes no bit of
// (tau, T, I), so the result is that of the lock-step march, bit for bit.
//   Lanes: a warp takes min(32, N_i) ADJACENT DIRECTIONS of one probe (and 32 / N_i neighbouring probes on cascades 0
// and 1).  Rays of a fan meet the same structure at nearly the same steps, so the lanes of a warp have similar work -
// with 32 probes of one direction (the lock-step mapping; 32-128 cells apart on the heavy cascades) a warp waited for
// its one lane inside a blob - and neighbouring lanes look up and gather neighbouring (often the same) cells.
//   Jump: after j steps the ray is at most j m + 2 cells (Chebyshev) from where it was, m = max(|wx|, |wy|) / (|wx| +
// |wy|) (j crossings of grid lines, shared between the axes in proportion, each count within one of its expectation);
// the cells closer than r are empty, so the steps before n + 1 + (r - 3)/m - and in any case before n + r, one cell per
// step - are skipped unseen.  Cascade 0's diagonals move one cell in x and y per step: m = 1.
//   The in-box prefix of the step table is not searched for: a ray ends at the first step outside the box.
// ------------------------------------------------------------------------------------------------
template <int LV, int WARPS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) march_fan_kernel(MarchParams p) {
    const int lane = threadIdx.x & 31;
    long long W = (long long)blockIdx.x * WARPS + (threadIdx.x >> 5);
    const long long ndir = 4LL * p.ngroups;
    const int ndl = (int)min(32LL, ndir), ppw = 32 / ndl;       // directions and probes per warp
    const long long nprobe = (long long)p.npx * p.npy;
    const long long ndb = ndir / ndl, npb = (nprobe + ppw - 1) / ppw;
    // warp order: direction block (fastest: the fans of one probe share cells near it), probe block, wavelength batch
    const long long db = W % ndb;
    W /= ndb;
    const long long pb = W % npb;
    const int nbI = (int)(W / npb);
    if (nbI >= p.nb) return;
    const long long k = db * ndl + (lane % ndl);
    const long long probe = pb * ppw + lane / ndl;
    bool valid = probe < nprobe;
    const int b = valid ? (int)(probe / p.npx) : 0, a = valid ? (int)(probe - (long long)b * p.npx) : 0;
    // a probe that is not flagged computes nothing and writes nothing; nothing flagged ever reads it
    if (valid && p.flags != nullptr) valid = __ldg(p.flags + probe) != 0;
    if (!__any_sync(FULL, valid)) return;
    const int half = (1 << p.shift) >> 1;
    const int X0 = (a << p.shift) + half, Y0 = (b << p.shift) + half;
    const long long ncell = (long long)p.nx * p.ny;
    const float *chiB = p.chiT + (long long)nbI * ncell * LV, *SB = p.ST + (long long)nbI * ncell * LV;

    float I[LV], tau[LV], T[LV];
#pragma unroll
    for (int v = 0; v < LV; v++) { I[v] = 0.f; tau[v] = 0.f; T[v] = 1.f; }
    unsigned nwalk = 0;
    if (p.cnt != nullptr && valid) {  // cnt == null: the cascade lies outside any box of this size (boundary term only)
        const long long o = __ldg(p.off + k);
        const int n = __ldg(p.cnt + k);
        const uint2 *tab = reinterpret_cast<const uint2 *>(p.steps + o);
        const unsigned *xyt = reinterpret_cast<const unsigned *>(p.xy + o);
        float invm = 1.f;
        if (p.cascade > 0) {
            float sw, cw;
            sincospif(2.f * ((float)k + 0.5f) / (float)ndir, &sw, &cw);
            sw = fabsf(sw); cw = fabsf(cw);
            invm = 0.999f * (sw + cw) / fmaxf(sw, cw);
        }
        int sn = 0;
        bool pend = false;
        float cP[LV], SP[LV], dsP = 0.f;
#pragma unroll
        for (int v = 0; v < LV; v++) { cP[v] = 0.f; SP[v] = 0.f; }
        // (cell, distance) of step sn when they have been looked up ahead of time: inside a blob the next step is the next
        // occupied cell, and its look-ups then overlap the integration of the previous one instead of following it
        bool ahead = false;
        int c_ahead = 0, r_ahead = 0;
        while (true) {
            bool found = false;
            int cf = 0;
            while (sn < n) {  // next occupied step of this lane's ray
                int r;
                if (ahead) {
                    cf = c_ahead; r = r_ahead; ahead = false;
                } else {
                    const unsigned e = __ldg(xyt + sn);
                    const int x = X0 + (int)(short)(e & 0xffffu), y = Y0 + (int)(short)(e >> 16);
                    if ((unsigned)x >= (unsigned)p.nx || (unsigned)y >= (unsigned)p.ny) { sn = n; break; }  // left the box: for good
                    cf = y * p.nx + x;
                    r = __ldg(p.dist + cf);
                }
                if (r == 0) { found = true; break; }
                sn += max(r, 1 + (int)((float)(r - 3) * invm));
            }
            float cN[LV], SN[LV], dsN = 0.f;
#pragma unroll
            for (int v = 0; v < LV; v++) { cN[v] = 0.f; SN[v] = 0.f; }
            if (found) {
                const unsigned long long d = (unsigned long long)cf * (LV * sizeof(float));
                load_vec<LV>(reinterpret_cast<const float *>(reinterpret_cast<const char *>(chiB) + d), cN);
                load_vec<LV>(reinterpret_cast<const float *>(reinterpret_cast<const char *>(SB) + d), SN);
                dsN = __uint_as_float(__ldg(tab + sn).y);
                sn++;
                if (sn < n) {  // look the next step up now
                    const unsigned e = __ldg(xyt + sn);
                    const int x = X0 + (int)(short)(e & 0xffffu), y = Y0 + (int)(short)(e >> 16);
                    if ((unsigned)x >= (unsigned)p.nx || (unsigned)y >= (unsigned)p.ny) {
                        sn = n;
                    } else {
                        c_ahead = y * p.nx + x;
                        r_ahead = __ldg(p.dist + c_ahead);
                        ahead = true;
                    }
                }
            }
            if (pend) {  // integrate the cell gathered one round earlier
                nwalk++;
                const float dkP = -dsP;
                if constexpr (LV >= 2) {
#pragma unroll
                    for (int q = 0; q < LV / 2; q++) {
                        f32x2 t2 = pk2(tau[2 * q], tau[2 * q + 1]), T2 = pk2(T[2 * q], T[2 * q + 1]), I2 = pk2(I[2 * q], I[2 * q + 1]);
                        seg_update2(pk2(cP[2 * q], cP[2 * q + 1]), pk2(SP[2 * q], SP[2 * q + 1]), pk2(dsP, dsP), pk2(dkP, dkP), t2, T2, I2);
                        up2(t2, tau[2 * q], tau[2 * q + 1]);
                        up2(T2, T[2 * q], T[2 * q + 1]);
                        up2(I2, I[2 * q], I[2 * q + 1]);
                    }
                } else {
                    seg_update1(cP[0], SP[0], dsP, tau[0], T[0], I[0]);
                }
                if (p.early_exit) {  // this ray is opaque at every wavelength: nothing more can arrive
                    float tmin = tau[0];
#pragma unroll
                    for (int v = 1; v < LV; v++) tmin = fminf(tmin, tau[v]);
                    if (tmin > p.tau_cut) { sn = n; found = false; ahead = false; }
                }
            }
            if (!found) break;  // per lane: nothing pending any more, nothing ahead
            pend = true;
            dsP = dsN;
#pragma unroll
            for (int v = 0; v < LV; v++) { cP[v] = cN[v]; SP[v] = SN[v]; }
        }
    }
    if (p.walked != nullptr) {
        unsigned long long mine = nwalk;
        for (int sh = 16; sh > 0; sh >>= 1) mine += __shfl_down_sync(FULL, mine, sh);
        if (lane == 0 && mine) atomicAdd(p.walked, mine);
    }
    // a2 (top cascade: boundary intensity) or a3 (bilinear parents, eq. 11): as in march_kernel
    if (valid) {
        if (p.Aup == nullptr) {
            const float *Ib = (2 * k < ndir) ? p.I_above : p.I_below;
#pragma unroll
            for (int v = 0; v < LV; v++) I[v] = fmaf(T[v], __ldg(Ib + nbI * LV + v), I[v]);
        } else {
            const int npxu = p.npx >> 1, npyu = p.npy >> 1;
            int a0, a1, b0, b1;
            float fa, fb;
            parent_axis(a, npxu, a0, a1, fa);
            parent_axis(b, npyu, b0, b1, fb);
            const float *up = p.Aup + (((long long)nbI * ndir + k) * npyu) * (long long)npxu * LV;
            float u00[LV], u01[LV], u10[LV], u11[LV];
            load_vec<LV>(up + ((long long)b0 * npxu + a0) * LV, u00);
            load_vec<LV>(up + ((long long)b0 * npxu + a1) * LV, u01);
            load_vec<LV>(up + ((long long)b1 * npxu + a0) * LV, u10);
            load_vec<LV>(up + ((long long)b1 * npxu + a1) * LV, u11);
#pragma unroll
            for (int v = 0; v < LV; v++) {
                const float lo = fmaf(fa, u01[v] - u00[v], u00[v]);
                const float hi = fmaf(fa, u11[v] - u10[v], u10[v]);
                I[v] = fmaf(T[v], fmaf(fb, hi - lo, lo), I[v]);
            }
        }
    }
    // mean over the 4 children of a direction group: 4 neighbouring lanes, added in child order like the lock-step march
    float acc[LV];
#pragma unroll
    for (int v = 0; v < LV; v++) {
        const float m1 = __shfl_down_sync(FULL, I[v], 1), m2 = __shfl_down_sync(FULL, I[v], 2), m3 = __shfl_down_sync(FULL, I[v], 3);
        acc[v] = 0.25f * ((((0.f + I[v]) + m1) + m2) + m3);
    }
    if (!valid || (lane & 3) != 0) return;
    const long long kg = k >> 2;
    if (p.mode == 0) {
        store_vec<LV>(p.out + (((long long)nbI * p.ngroups + kg) * nprobe + probe) * LV, acc);
    } else if (p.mode == 1) {  // cascade 0: a4, J
        float *o = p.out + probe * p.L + nbI * LV;
        if ((nbI + 1) * LV <= p.L && (p.L % LV) == 0) {
            store_vec<LV>(o, acc);
        } else {
#pragma unroll
            for (int v = 0; v < LV; v++)
                if (nbI * LV + v < p.L) o[v] = acc[v];
        }
    } else {
        float sum = 0.f;
#pragma unroll
        for (int v = 0; v < LV; v++) sum = fmaf(__ldg(p.weights + nbI * LV + v), acc[v], sum);
        p.out[(long long)nbI * nprobe + probe] = sum;
    }
}

template <int LV>
static cudaError_t launch_march_sparse(const MarchParams &p, cudaStream_t st) {
    constexpr int WARPS = 8;
    const long long ndir = 4LL * p.ngroups, ndl = ndir < 32 ? ndir : 32, ppw = 32 / ndl;
    const long long nprobe = (long long)p.npx * p.npy;
    const long long warps = (ndir / ndl) * ((nprobe + ppw - 1) / ppw) * p.nb;
    const long long blocks = (warps + WARPS - 1) / WARPS;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (blocks == 0) return cudaSuccess;
    // sparse_mode: blocks of 8 / 4 / 2 warps at <= 80 registers (24 warps/SM; a block keeps its slots until its last warp
    // is done, and the work of a warp depends on what its fan meets), or 3: blocks of 4 warps at <= 128 registers (16 warps/SM)
    switch (p.sparse_mode) {
        case 1: march_fan_kernel<LV, 4, 6><<<(unsigned)((warps + 3) / 4), 128, 0, st>>>(p); break;
        case 2: march_fan_kernel<LV, 2, 12><<<(unsigned)((warps + 1) / 2), 64, 0, st>>>(p); break;
        case 3: march_fan_kernel<LV, 4, 4><<<(unsigned)((warps + 3) / 4), 128, 0, st>>>(p); break;
        default: march_fan_kernel<LV, WARPS, 3><<<(unsigned)blocks, WARPS * 32, 0, st>>>(p); break;
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Hit lists (mostly empty atmospheres, built by rc_analyse_atmosphere when the caller lends room for them): which steps
// of a ray meet an occupied cell depends on the geometry and the occupancy alone - not on the wavelength, not on the
// values.  The fan march finds them again for every wavelength batch of every solve (half of its time on config 4);
// here they are found once: per cascade, hit_off[ray] .. hit_off[ray + 1] index the ray's occupied in-box steps (their
// numbers in the direction's step table, uint16) in hit_list, ray = probe * N_i + k.  march_list_kernel then only
// gathers and integrates - the same cells in the same order as the fan and the lock-step march: bit-identical.
// ------------------------------------------------------------------------------------------------
// 32 rays per warp (a fan of adjacent directions of one probe, as march_fan_kernel).  FILL = false: cnt[ray] = number of
// hits (and *total += them); FILL = true: list[off[ray] + i] = step of the i-th hit.
template <bool FILL>
__global__ void __launch_bounds__(256) hit_walk_kernel(MarchParams p, unsigned *cnt_or_off, unsigned short *list, unsigned long long *total) {
    const int lane = threadIdx.x & 31;
    long long W = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long ndir = 4LL * p.ngroups;
    const int ndl = (int)min(32LL, ndir), ppw = 32 / ndl;
    const long long nprobe = (long long)p.npx * p.npy;
    const long long ndb = ndir / ndl, npb = (nprobe + ppw - 1) / ppw;
    if (W >= ndb * npb) return;
    const long long db = W % ndb, pb = W / ndb;
    const long long k = db * ndl + (lane % ndl);
    const long long probe = pb * ppw + lane / ndl;
    bool valid = probe < nprobe;
    const int b = valid ? (int)(probe / p.npx) : 0, a = valid ? (int)(probe - (long long)b * p.npx) : 0;
    if (valid && p.flags != nullptr) valid = __ldg(p.flags + probe) != 0;
    const int half = (1 << p.shift) >> 1;
    const int X0 = (a << p.shift) + half, Y0 = (b << p.shift) + half;
    unsigned nhit = 0;
    if (p.cnt != nullptr && valid) {
        const long long o = __ldg(p.off + k);
        const int n = __ldg(p.cnt + k);
        const unsigned *xyt = reinterpret_cast<const unsigned *>(p.xy + o);
        float invm = 1.f;
        if (p.cascade > 0) {  // the same jump rule as march_fan_kernel
            float sw, cw;
            sincospif(2.f * ((float)k + 0.5f) / (float)ndir, &sw, &cw);
            sw = fabsf(sw); cw = fabsf(cw);
            invm = 0.999f * (sw + cw) / fmaxf(sw, cw);
        }
        unsigned short *out = nullptr;
        if constexpr (FILL) out = list + __ldg(cnt_or_off + probe * ndir + k);
        int sn = 0;
        while (sn < n) {
            const unsigned e = __ldg(xyt + sn);
            const int x = X0 + (int)(short)(e & 0xffffu), y = Y0 + (int)(short)(e >> 16);
            if ((unsigned)x >= (unsigned)p.nx || (unsigned)y >= (unsigned)p.ny) break;  // left the box: for good
            const int r = __ldg(p.dist + (long long)y * p.nx + x);
            if (r == 0) {
                if constexpr (FILL) out[nhit] = (unsigned short)sn;
                nhit++;
                sn++;
            } else {
                sn += max(r, 1 + (int)((float)(r - 3) * invm));
            }
        }
    }
    if constexpr (!FILL) {
        if (probe < nprobe && cnt_or_off != nullptr) cnt_or_off[probe * ndir + k] = nhit;
        unsigned long long mine = nhit;
        for (int sh = 16; sh > 0; sh >>= 1) mine += __shfl_down_sync(FULL, mine, sh);
        if (lane == 0 && mine) atomicAdd(total, mine);
    }
}

// Exclusive prefix sum of n counts, in place (a[n] = the total): per-block sums, one block over those, add back.
__global__ void __launch_bounds__(1024) scan_block_kernel(unsigned *a, long long n, unsigned *bsum) {
    __shared__ unsigned ws[32];
    const long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
    const unsigned v = i < n ? a[i] : 0u;
    unsigned x = v;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int sh = 1; sh < 32; sh <<= 1) { const unsigned y = __shfl_up_sync(FULL, x, sh); if (lane >= sh) x += y; }
    if (lane == 31) ws[w] = x;
    __syncthreads();
    if (w == 0) {
        unsigned t = ws[lane];
        for (int sh = 1; sh < 32; sh <<= 1) { const unsigned y = __shfl_up_sync(FULL, t, sh); if (lane >= sh) t += y; }
        ws[lane] = t;
    }
    __syncthreads();
    const unsigned incl = x + (w > 0 ? ws[w - 1] : 0u);
    if (i < n) a[i] = incl - v;  // exclusive within the block
    if (threadIdx.x == 1023) bsum[blockIdx.x] = incl;
}

__global__ void __launch_bounds__(1024) scan_sums_kernel(unsigned *bsum, int nblocks) {  // one block: exclusive scan of the block sums
    __shared__ unsigned ws[32];
    __shared__ unsigned carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int start = 0; start < nblocks; start += 1024) {
        const int i = start + threadIdx.x;
        const unsigned v = i < nblocks ? bsum[i] : 0u;
        unsigned x = v;
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        for (int sh = 1; sh < 32; sh <<= 1) { const unsigned y = __shfl_up_sync(FULL, x, sh); if (lane >= sh) x += y; }
        if (lane == 31) ws[w] = x;
        __syncthreads();
        if (w == 0) {
            unsigned t = ws[lane];
            for (int sh = 1; sh < 32; sh <<= 1) { const unsigned y = __shfl_up_sync(FULL, t, sh); if (lane >= sh) t += y; }
            ws[lane] = t;
        }
        __syncthreads();
        const unsigned incl = x + (w > 0 ? ws[w - 1] : 0u) + carry;
        if (i < nblocks) bsum[i] = incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry = incl;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(1024) scan_add_kernel(unsigned *a, long long n, const unsigned *bsum, unsigned long long total) {
    const long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
    if (i < n) a[i] += bsum[blockIdx.x];
    if (i == n) a[n] = (unsigned)total;
}

// *flag = 1 if the two occupancy maps differ anywhere (hit lists are kept while the occupancy they were built for stands)
__global__ void occ_differs_kernel(const unsigned char *a, const unsigned char *b, long long n, int *flag) {
    bool d = false;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) d = d || a[i] != b[i];
    if (__any_sync(FULL, d) && (threadIdx.x & 31) == 0) *flag = 1;
}

cudaError_t launch_occ_differs(const unsigned char *a, const unsigned char *b, long long n, int *flag, cudaStream_t st) {
    occ_differs_kernel<<<148 * 4, 256, 0, st>>>(a, b, n, flag);
    return cudaGetLastError();
}

// counts -> offsets for one cascade; `total` (host) must be the sum already known from the counting pass
cudaError_t launch_hit_scan(unsigned *a, long long n, unsigned *bsum, unsigned long long total, cudaStream_t st) {
    const long long nblocks = (n + 1023) / 1024;
    scan_block_kernel<<<(unsigned)nblocks, 1024, 0, st>>>(a, n, bsum);
    scan_sums_kernel<<<1, 1024, 0, st>>>(bsum, (int)nblocks);
    scan_add_kernel<<<(unsigned)((n + 1 + 1023) / 1024), 1024, 0, st>>>(a, n, bsum, total);
    return cudaGetLastError();
}

cudaError_t launch_hit_walk(const MarchParams &p, bool fill, unsigned *cnt_or_off, unsigned short *list, unsigned long long *total, cudaStream_t st) {
    const long long ndir = 4LL * p.ngroups, ndl = ndir < 32 ? ndir : 32, ppw = 32 / ndl;
    const long long nprobe = (long long)p.npx * p.npy;
    const long long warps = (ndir / ndl) * ((nprobe + ppw - 1) / ppw);
    const long long blocks = (warps + 7) / 8;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (fill) hit_walk_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(p, cnt_or_off, list, total);
    else hit_walk_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(p, cnt_or_off, list, total);
    return cudaGetLastError();
}

// The march over hit lists.  A warp = R = 32 / B adjacent directions of one probe (or of R / N_i probes on cascades 0, 1) x
// B wavelength batches: the B lanes of a ray read the same list entries and table steps (one sector, broadcast) and gather
// B x LV consecutive floats of the cell (under this march the packed arrays are [batch group][cell][batch in group][LV]).  The next
// hit's step, cell and path length are looked up while the previous cell is integrated.
template <int LV, int NM, int B, int WARPS, int MINB, bool LINE>
__global__ void __launch_bounds__(WARPS * 32, MINB) march_list_kernel(MarchParams p) {
    constexpr int R = 32 / B;
    constexpr int LL = LV / NM;  // wavelengths per lane; channel ch = l * NM + m (2.5D: NM inclinations per wavelength)
    const int lane = threadIdx.x & 31;
    long long W = (long long)blockIdx.x * WARPS + (threadIdx.x >> 5);
    const long long ndir = 4LL * p.ngroups;
    const int ndl = (int)min((long long)R, ndir), ppw = R / ndl;  // directions and probes per warp
    const long long nprobe = (long long)p.npx * p.npy;
    const long long ndb = ndir / ndl, npb = (nprobe + ppw - 1) / ppw;
    const int nbg = (p.nb + B - 1) / B;
    const long long db = W % ndb;
    W /= ndb;
    const long long pb = W % npb;
    const int bg = (int)(W / npb);
    if (bg >= nbg) return;
    const int r = lane / B, nbI = bg * B + lane % B;
    const long long k = db * ndl + (r % ndl);
    const long long probe = pb * ppw + r / ndl;
    bool valid = probe < nprobe && nbI < p.nb;
    const int b = probe < nprobe ? (int)(probe / p.npx) : 0, a = probe < nprobe ? (int)(probe - (long long)b * p.npx) : 0;
    if (valid && p.flags != nullptr) valid = __ldg(p.flags + probe) != 0;
    if (!__any_sync(FULL, valid)) return;
    const int half = (1 << p.shift) >> 1;
    const int X0 = (a << p.shift) + half, Y0 = (b << p.shift) + half;
    // packed arrays: [batch group][cell][batch in group][LL]; LINE: the six packed line parameters of the cell, [cell][6]
    // (the same 24 bytes for every lane of the ray), opacity and source function evaluated per ray as in march_kernel
    constexpr int NR = LINE ? 6 : LL;
    const int Bg = min(B, p.nb - bg * B);
    const long long gbase = LINE ? 0 : ((long long)bg * B * ((long long)p.nx * p.ny) + (nbI - bg * B)) * LL;
    const float *chiB = LINE ? p.linepk : p.chiT + gbase, *SB = LINE ? nullptr : p.ST + gbase;  // + cell * Bg * LL
    const unsigned long long cstride = LINE ? 24ull : (unsigned long long)Bg * (LL * sizeof(float));
    float xs[LINE ? LL : 1], wx = 0.f, wy = 0.f;
    if constexpr (LINE) {
#pragma unroll
        for (int v = 0; v < LL; v++) xs[v] = __ldg(p.xls + min(nbI, p.nb - 1) * LL + v);
        sincospif(2.f * ((float)k + 0.5f) / (float)ndir, &wy, &wx);
    }

    float I[LV], tau[LV], T[LV];
#pragma unroll
    for (int v = 0; v < LV; v++) { I[v] = 0.f; tau[v] = 0.f; T[v] = 1.f; }
    unsigned nwalk = 0;
    if (p.cnt != nullptr && valid) {
        const long long o = __ldg(p.off + k);
        const uint2 *tab = reinterpret_cast<const uint2 *>(p.steps + o);
        const unsigned *xyt = reinterpret_cast<const unsigned *>(p.xy + o);
        const unsigned h0 = __ldg(p.hit_off + probe * ndir + k), h1 = __ldg(p.hit_off + probe * ndir + k + 1);
        const unsigned short *hl = p.hit_list;
        // three stages in flight: the step number two hits ahead, (cell, ds) one hit ahead, (chi, S) of the hit being integrated
        unsigned h = h0;
        int s2 = h < h1 ? (int)__ldg(hl + h) : -1;
        h++;
        int c1 = -1;
        float d1 = 0.f;
        auto lookup = [&]() {  // stage 2 <- stage 1; stage 1 <- list
            if (s2 >= 0) {
                const unsigned e = __ldg(xyt + s2);
                c1 = (Y0 + (int)(short)(e >> 16)) * p.nx + X0 + (int)(short)(e & 0xffffu);
                d1 = __uint_as_float(__ldg(tab + s2).y);
            } else {
                c1 = -1;
            }
            s2 = h < h1 ? (int)__ldg(hl + h) : -1;
            h++;
        };
        lookup();
        float cP[NR], SP[LINE ? 1 : LL], dsP = 0.f;
        bool pend = false;
        while (true) {
            float cN[NR], SN[LINE ? 1 : LL];
            const bool have = c1 >= 0;
            const float dsN = d1;
            if (have) {
                const unsigned long long d = (unsigned long long)(unsigned)c1 * cstride;
                if constexpr (LINE) {
                    const float2 *src = reinterpret_cast<const float2 *>(reinterpret_cast<const char *>(chiB) + d);
                    const float2 q0 = __ldg(src), q1 = __ldg(src + 1), q2 = __ldg(src + 2);
                    cN[0] = q0.x; cN[1] = q0.y; cN[2] = q1.x; cN[3] = q1.y; cN[4] = q2.x; cN[5] = q2.y;
                } else {
                    load_vec<LL>(reinterpret_cast<const float *>(reinterpret_cast<const char *>(chiB) + d), cN);
                    load_vec<LL>(reinterpret_cast<const float *>(reinterpret_cast<const char *>(SB) + d), SN);
                }
                lookup();
            }
            bool stop = !have;
            if (pend) {  // integrate the cell gathered one round earlier
                nwalk++;
                float dsm[NM];  // inclination m crosses the same cell over ds / sin(inclination)
#pragma unroll
                for (int m = 0; m < NM; m++) dsm[m] = NM == 1 ? dsP : dsP * p.incl_f[m];
                if constexpr (LINE) {
                    // a = x_l + v.w (photons travel along -w), inclination m sees the in-plane velocity times sin(inclination)
                    const float vw = fmaf(cP[4], wx, cP[5] * wy);
                    float vwm[NM], dkm[NM];
#pragma unroll
                    for (int m = 0; m < NM; m++) { vwm[m] = NM == 1 ? vw : vw * p.incl_s[m]; dkm[m] = dsm[m] * KAPPA; }
                    if constexpr (LV >= 2) {
#pragma unroll
                        for (int q = 0; q < LV / 2; q++) {
                            const int lo = LL >= 2 ? (2 * (q / NM)) * NM + q % NM : 2 * q, hi = LL >= 2 ? (2 * (q / NM) + 1) * NM + q % NM : 2 * q + 1;
                            const int l0 = LL >= 2 ? 2 * (q / NM) : 0, l1 = LL >= 2 ? l0 + 1 : 0;
                            const int m0 = LL >= 2 ? q % NM : 2 * q, m1 = LL >= 2 ? m0 : 2 * q + 1;
                            f32x2 t2 = pk2(tau[lo], tau[hi]), T2 = pk2(T[lo], T[hi]), I2 = pk2(I[lo], I[hi]);
                            seg_update_line2(add2(pk2(xs[l0], xs[l1]), pk2(vwm[m0], vwm[m1])), cP[0], cP[1], cP[2], cP[3],
                                             pk2(dsm[m0], dsm[m1]), pk2(dkm[m0], dkm[m1]), t2, T2, I2);
                            up2(t2, tau[lo], tau[hi]);
                            up2(T2, T[lo], T[hi]);
                            up2(I2, I[lo], I[hi]);
                        }
                    } else {
                        const float aa = xs[0] + vwm[0];
                        const float phi = ex2_neg(aa * aa);
                        seg_update_line(fmaf(cP[2], phi, cP[0]), fmaf(cP[3], phi, cP[1]), dsm[0], dkm[0], tau[0], T[0], I[0]);
                    }
                } else if constexpr (LV >= 2) {
#pragma unroll
                    for (int q = 0; q < LV / 2; q++) {  // the pairs of march_kernel: two wavelengths of one inclination, or (LL = 1) two inclinations
                        const int lo = LL >= 2 ? (2 * (q / NM)) * NM + q % NM : 2 * q, hi = LL >= 2 ? (2 * (q / NM) + 1) * NM + q % NM : 2 * q + 1;
                        const int l0 = LL >= 2 ? 2 * (q / NM) : 0, l1 = LL >= 2 ? l0 + 1 : 0;
                        const int m0 = LL >= 2 ? q % NM : 2 * q, m1 = LL >= 2 ? m0 : 2 * q + 1;
                        f32x2 t2 = pk2(tau[lo], tau[hi]), T2 = pk2(T[lo], T[hi]), I2 = pk2(I[lo], I[hi]);
                        seg_update2(pk2(cP[l0], cP[l1]), pk2(SP[l0], SP[l1]), pk2(dsm[m0], dsm[m1]), pk2(-dsm[m0], -dsm[m1]), t2, T2, I2);
                        up2(t2, tau[lo], tau[hi]);
                        up2(T2, T[lo], T[hi]);
                        up2(I2, I[lo], I[hi]);
                    }
                } else {
                    seg_update1(cP[0], SP[0], dsP, tau[0], T[0], I[0]);
                }
                if (p.early_exit) {  // this ray is opaque at every wavelength of the lane: nothing more can arrive
                    float tmin = tau[0];
#pragma unroll
                    for (int v = 1; v < LV; v++) tmin = fminf(tmin, tau[v]);
                    if (tmin > p.tau_cut) stop = true;
                }
            }
            if (stop) break;
            pend = true;
            dsP = dsN;
#pragma unroll
            for (int v = 0; v < NR; v++) cP[v] = cN[v];
            if constexpr (!LINE) {
#pragma unroll
                for (int v = 0; v < LL; v++) SP[v] = SN[v];
            }
        }
    }
    if (p.walked != nullptr) {
        unsigned long long mine = nwalk;
        for (int sh = 16; sh > 0; sh >>= 1) mine += __shfl_down_sync(FULL, mine, sh);
        if (lane == 0 && mine) atomicAdd(p.walked, mine);
    }
    // a2 / a3 as in march_kernel
    if (valid) {
        if (p.Aup == nullptr) {
            const float *Ib = (2 * k < ndir) ? p.I_above : p.I_below;
#pragma unroll
            for (int v = 0; v < LV; v++) I[v] = fmaf(T[v], __ldg(Ib + nbI * LV + v), I[v]);
        } else {
            const int npxu = p.npx >> 1, npyu = p.npy >> 1;
            int a0, a1, b0, b1;
            float fa, fb;
            parent_axis(a, npxu, a0, a1, fa);
            parent_axis(b, npyu, b0, b1, fb);
            const float *up = p.Aup + (((long long)nbI * ndir + k) * npyu) * (long long)npxu * LV;
            float u00[LV], u01[LV], u10[LV], u11[LV];
            load_vec<LV>(up + ((long long)b0 * npxu + a0) * LV, u00);
            load_vec<LV>(up + ((long long)b0 * npxu + a1) * LV, u01);
            load_vec<LV>(up + ((long long)b1 * npxu + a0) * LV, u10);
            load_vec<LV>(up + ((long long)b1 * npxu + a1) * LV, u11);
#pragma unroll
            for (int v = 0; v < LV; v++) {
                const float lo = fmaf(fa, u01[v] - u00[v], u00[v]);
                const float hi = fmaf(fa, u11[v] - u10[v], u10[v]);
                I[v] = fmaf(T[v], fmaf(fb, hi - lo, lo), I[v]);
            }
        }
    }
    // mean over the 4 children of a direction group: lanes B apart, added in child order like the lock-step march
    float acc[LV];
#pragma unroll
    for (int v = 0; v < LV; v++) {
        const float m1 = __shfl_down_sync(FULL, I[v], B), m2 = __shfl_down_sync(FULL, I[v], 2 * B), m3 = __shfl_down_sync(FULL, I[v], 3 * B);
        acc[v] = 0.25f * ((((0.f + I[v]) + m1) + m2) + m3);
    }
    if (!valid || (r & 3) != 0) return;
    const long long kg = k >> 2;
    if (p.mode == 0) {
        store_vec<LV>(p.out + (((long long)nbI * p.ngroups + kg) * nprobe + probe) * LV, acc);
    } else {
        // cascade 0: J_l = sum over the inclinations of w_m x (mean of the 4 directions)  (a4)
        float Jl[LL];
#pragma unroll
        for (int l = 0; l < LL; l++) {
            Jl[l] = NM == 1 ? acc[l] : 0.f;
            if constexpr (NM > 1) {
#pragma unroll
                for (int m = 0; m < NM; m++) Jl[l] = fmaf(p.incl_w[m], acc[l * NM + m], Jl[l]);
            }
        }
        if (p.mode == 1) {
            float *o = p.out + probe * p.L + nbI * LL;
            if ((nbI + 1) * LL <= p.L && (p.L % LL) == 0) {
                store_vec<LL>(o, Jl);
            } else {
#pragma unroll
                for (int v = 0; v < LL; v++)
                    if (nbI * LL + v < p.L) o[v] = Jl[v];
            }
        } else {
            float sum = 0.f;
#pragma unroll
            for (int v = 0; v < LL; v++) sum = fmaf(__ldg(p.weights + nbI * LL + v), Jl[v], sum);
            p.out[(long long)nbI * nprobe + probe] = sum;
        }
    }
}

template <int LV, int NM, int B, bool LINE>
static cudaError_t launch_march_list_b(const MarchParams &p, cudaStream_t st) {
    constexpr int R = 32 / B;
    const long long ndir = 4LL * p.ngroups, ndl = ndir < R ? ndir : R, ppw = R / ndl;
    const long long nprobe = (long long)p.npx * p.npy;
    const long long warps = (ndir / ndl) * ((nprobe + ppw - 1) / ppw) * ((p.nb + B - 1) / B);
    if ((warps + 3) / 4 > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (warps == 0) return cudaSuccess;
    if constexpr (NM == 1 && !LINE) {
        switch (p.sparse_mode) {  // blocks of 4 warps at <= 80 / 96 / 128 registers (24 / 20 / 16 warps per SM), or 8 warps at <= 80
            case 0: march_list_kernel<LV, NM, B, 8, 3, false><<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(p); return cudaGetLastError();
            case 2: march_list_kernel<LV, NM, B, 4, 5, false><<<(unsigned)((warps + 3) / 4), 128, 0, st>>>(p); return cudaGetLastError();
            case 3: march_list_kernel<LV, NM, B, 4, 4, false><<<(unsigned)((warps + 3) / 4), 128, 0, st>>>(p); return cudaGetLastError();
            default: break;
        }
    }
    march_list_kernel<LV, NM, B, 4, 6, LINE><<<(unsigned)((warps + 3) / 4), 128, 0, st>>>(p);
    return cudaGetLastError();
}

template <int LV, int NM, bool LINE>
static cudaError_t launch_march_list_l(const MarchParams &p, cudaStream_t st) {
    switch (p.list_b) {
        case 8: return launch_march_list_b<LV, NM, 8, LINE>(p, st);
        case 4: return launch_march_list_b<LV, NM, 4, LINE>(p, st);
        case 2: return launch_march_list_b<LV, NM, 2, LINE>(p, st);
        default: return launch_march_list_b<LV, NM, 1, LINE>(p, st);
    }
}

template <int LV, int NM = 1>
static cudaError_t launch_march_list(const MarchParams &p, cudaStream_t st) {
    return p.linepk != nullptr ? launch_march_list_l<LV, NM, true>(p, st) : launch_march_list_l<LV, NM, false>(p, st);
}

// Velocity-dependent line mode (linepk != null): 3 MUFU per segment-channel, ring of 2, 24 warps/SM.
template <int LV, int NM = 1>
static cudaError_t launch_march_line(const MarchParams &p, cudaStream_t st) {
    constexpr int WARPS = 8;
    const long long blocks = (march_warps(p) + WARPS - 1) / WARPS;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (blocks == 0) return cudaSuccess;
    march_kernel<LV, NM, 2, WARPS, 3, false, true><<<(unsigned)blocks, WARPS * 32, 0, st>>>(p);
    return cudaGetLastError();
}

template <int LV>
static cudaError_t launch_march_flat(const MarchParams &p, int variant, cudaStream_t st) {
    if (p.hit_list != nullptr) return launch_march_list<LV>(p, st);  // (flat or moving line)
    if (p.linepk != nullptr) return launch_march_line<LV>(p, st);
    if (p.dist != nullptr) return launch_march_sparse<LV>(p, st);
    switch (variant) {
        case 0: return launch_march_variant<LV, 1, 2, 8, 3>(p, st);
        case 1: return launch_march_variant<LV, 1, 3, 4, 5>(p, st);
        case 3: return launch_march_variant<LV, 1, 4, 8, 2>(p, st);
        case 4: return launch_march_variant<LV, 1, 2, 4, 5>(p, st);
        default: return launch_march_variant<LV, 1, 3, 8, 2>(p, st);
    }
}

// LV = channels per lane = (wavelengths per lane) x NM inclinations; the inclined launches come in one
// variant only
cudaError_t launch_march(const MarchParams &p, int LV, int NM, int variant, cudaStream_t st) {
    if (NM == 1) {
        switch (LV) {
            case 8: return launch_march_flat<8>(p, variant, st);
            case 4: return launch_march_flat<4>(p, variant, st);
            case 2: return launch_march_flat<2>(p, variant, st);
            default: return launch_march_flat<1>(p, variant, st);
        }
    }
    if (p.hit_list != nullptr) {  // the sparse march over hit lists, inclined (flat or moving line)
        switch (LV * 16 + NM) {
            case 8 * 16 + 8: return launch_march_list<8, 8>(p, st);
            case 8 * 16 + 4: return launch_march_list<8, 4>(p, st);
            case 8 * 16 + 2: return launch_march_list<8, 2>(p, st);
            case 4 * 16 + 4: return launch_march_list<4, 4>(p, st);
            case 4 * 16 + 2: return launch_march_list<4, 2>(p, st);
            case 2 * 16 + 2: return launch_march_list<2, 2>(p, st);
            default: return cudaErrorInvalidValue;
        }
    }
    if (p.linepk != nullptr) {
        switch (LV * 16 + NM) {
            case 8 * 16 + 8: return launch_march_line<8, 8>(p, st);
            case 8 * 16 + 4: return launch_march_line<8, 4>(p, st);
            case 8 * 16 + 2: return launch_march_line<8, 2>(p, st);
            case 4 * 16 + 4: return launch_march_line<4, 4>(p, st);
            case 4 * 16 + 2: return launch_march_line<4, 2>(p, st);
            case 2 * 16 + 2: return launch_march_line<2, 2>(p, st);
            default: return cudaErrorInvalidValue;
        }
    }
    // inclined launches are MUFU-bound (NM ex2 per gathered value): ring of 2, 24 warps/SM measured best
    switch (LV * 16 + NM) {
        case 8 * 16 + 8: return launch_march_variant<8, 8, 2, 8, 3>(p, st);
        case 8 * 16 + 4: return launch_march_variant<8, 4, 2, 8, 3>(p, st);
        case 8 * 16 + 2: return launch_march_variant<8, 2, 2, 8, 3>(p, st);
        case 4 * 16 + 4: return launch_march_variant<4, 4, 2, 8, 3>(p, st);
        case 4 * 16 + 2: return launch_march_variant<4, 2, 2, 8, 3>(p, st);
        case 2 * 16 + 2: return launch_march_variant<2, 2, 2, 8, 3>(p, st);
        default: return cudaErrorInvalidValue;
    }
}

// ------------------------------------------------------------------------------------------------
// Jbar = sum over wavelength batches of the per-batch weighted sums (deterministic order).
// ------------------------------------------------------------------------------------------------
__global__ void reduce_jbar_kernel(const float *Jpart, float *Jbar, long long ncell, int nb) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    float s = 0.f;
    for (int b = 0; b < nb; b++) s += Jpart[(long long)b * ncell + c];
    Jbar[c] = s;
}

cudaError_t launch_reduce_jbar(const float *Jpart, float *Jbar, long long ncell, int nb, cudaStream_t st) {
    reduce_jbar_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, st>>>(Jpart, Jbar, ncell, nb);
    return cudaGetLastError();
}

// RC_VALIDATE: flag |= 1 if any chi/eta is negative or non-finite.
__global__ void validate_kernel(const float *chi, const float *eta, long long n, int *flag) {
    int bad = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const float c = chi[i], e = eta[i];
        if (!(c >= 0.f) || !(e >= 0.f) || isinf(c) || isinf(e)) bad |= 1;
    }
    if (bad) atomicOr(flag, bad);
}

// Marks the cells that hold a non-zero value (coalesced over the whole array).  W floats per thread: 4 when the
// row width is a multiple of 4, else 1; `posmask`: bit (position within the cell's row, mod 32) set = position counts
// (all of chi / eta; in line mode positions 0 and 2 of the six parameters, chi_c and chi_line).
template <int W>
__global__ void mark_occupied_kernel(const float *f, long long nchunk, int chunks_per_cell, int *mark, unsigned posmask) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nchunk; i += (long long)gridDim.x * blockDim.x) {
        bool nz;
        if constexpr (W == 4) {
            const float4 v = __ldg(reinterpret_cast<const float4 *>(f) + i);
            nz = v.x != 0.f || v.y != 0.f || v.z != 0.f || v.w != 0.f;
        } else {
            nz = __ldg(f + i) != 0.f && (chunks_per_cell > 32 || ((posmask >> (unsigned)(i % chunks_per_cell)) & 1u));
        }
        if (nz) mark[i / chunks_per_cell] = 1;
    }
}

cudaError_t launch_validate(const float *chi, const float *eta, long long n, int *flag, cudaStream_t st) {
    validate_kernel<<<148 * 8, 256, 0, st>>>(chi, eta, n, flag);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Sparsity as the paper defines it: "this flag then defines the probes of cascade 0 that may be involved
// ... Their bilinear "parents" are recursively flagged up to the maximum cascade, and the radiance intervals are only
// computed for these flagged probes".
// ------------------------------------------------------------------------------------------------
// flag[0] = the cells of interest (any non-zero byte), as 0 / 1
__global__ void flags_from_active_kernel(const unsigned char *active, unsigned char *flag0, long long ncell) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < ncell) flag0[c] = active[c] != 0;
}

// every flagged probe of cascade i flags its four bilinear parents in cascade i+1 (stores of the same value: no race)
__global__ void flag_parents_kernel(const unsigned char *child, int npx, int npy, unsigned char *parent) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= (long long)npx * npy || child[c] == 0) return;
    const int b = (int)(c / npx), a = (int)(c - (long long)b * npx), upx = npx >> 1, upy = npy >> 1;
    int a0, a1, b0, b1;
    float f;
    parent_axis(a, upx, a0, a1, f);
    parent_axis(b, upy, b0, b1, f);
    parent[(long long)b0 * upx + a0] = 1; parent[(long long)b0 * upx + a1] = 1;
    parent[(long long)b1 * upx + a0] = 1; parent[(long long)b1 * upx + a1] = 1;
}

// one warp per patch of the march's own warp -> probe mapping (warp_work): does the patch hold a flagged probe?
__global__ void mark_patches_kernel(MarchParams p, unsigned char *mark, int npatch) {
    const int lane = threadIdx.x & 31;
    const long long W = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (W >= npatch) return;
    // p arrives with kg_n = ngroups, nb = 1, cpw = 0, plist = null: warp W * G is direction group 0 of patch W
    const WarpWork ww = warp_work(p, W * min(p.kg_n, 8), lane);
    const unsigned any = __ballot_sync(FULL, ww.valid);
    if (lane == 0) mark[W] = any != 0u;
}

// ordered compaction of the marked patch numbers by one block (setup time only): list[0 .. *count)
__global__ void __launch_bounds__(1024) compact_patches_kernel(const unsigned char *mark, int n, int *list, int *count) {
    __shared__ int wsum[32];
    __shared__ int base;
    if (threadIdx.x == 0) base = 0;
    __syncthreads();
    for (int start = 0; start < n; start += 1024) {
        const int i = start + threadIdx.x;
        const int m = i < n && mark[i] != 0;
        const unsigned bal = __ballot_sync(FULL, m);
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        if (lane == 0) wsum[w] = __popc(bal);
        __syncthreads();
        int off = base;
        for (int q = 0; q < w; q++) off += wsum[q];
        if (m) list[off + __popc(bal & ((1u << lane) - 1u))] = i;
        __syncthreads();
        if (threadIdx.x == 0) {
            int t = 0;
            for (int q = 0; q < 32; q++) t += wsum[q];
            base += t;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) *count = base;
}

// *out += the number of non-zero bytes of a[0 .. n): the flagged probes of one cascade, for rc_stats
__global__ void __launch_bounds__(256) count_flags_kernel(const unsigned char *a, long long n, unsigned long long *out) {
    unsigned mine = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) mine += a[i] != 0;
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_down_sync(FULL, mine, o);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(out, (unsigned long long)mine);
}

cudaError_t launch_count_flags(const unsigned char *a, long long n, unsigned long long *out, cudaStream_t st) {
    const long long want = (n + 255) / 256;
    count_flags_kernel<<<(unsigned)(want < 148 * 8 ? want : 148 * 8), 256, 0, st>>>(a, n, out);
    return cudaGetLastError();
}

cudaError_t launch_flags_from_active(const unsigned char *active, unsigned char *flag0, long long ncell, cudaStream_t st) {
    flags_from_active_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, st>>>(active, flag0, ncell);
    return cudaGetLastError();
}

cudaError_t launch_flag_parents(const unsigned char *child, int npx, int npy, unsigned char *parent, cudaStream_t st) {
    const long long n = (long long)npx * npy;
    flag_parents_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(child, npx, npy, parent);
    return cudaGetLastError();
}

cudaError_t launch_mark_and_compact_patches(const MarchParams &p, int npatch, unsigned char *mark, int *list, int *count, cudaStream_t st) {
    mark_patches_kernel<<<(unsigned)(((long long)npatch * 32 + 255) / 256), 256, 0, st>>>(p, mark, npatch);
    compact_patches_kernel<<<1, 1024, 0, st>>>(mark, npatch, list, count);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Free-space acceleration: occupancy of the cells (flagged, and chi or eta non-zero at some
// wavelength) and its Chebyshev distance transform, clamped at 255: dist = 0 on an occupied cell, else the distance to
// the nearest one.  Setup time only; separable brute force with early termination.
// ------------------------------------------------------------------------------------------------
__global__ void occupancy_kernel(const int *mark, const unsigned char *active, unsigned char *occ, long long ncell, unsigned long long *nempty) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    bool e = false;
    if (c < ncell) {
        const bool o = mark[c] != 0 && (active == nullptr || active[c] != 0);
        occ[c] = o;
        e = !o;
    }
    const unsigned bal = __ballot_sync(FULL, e);
    if ((threadIdx.x & 31) == 0 && bal) atomicAdd(nempty, (unsigned long long)__popc(bal));
}

// d1[y][x] = distance along the row to the nearest occupied cell of row y (255: none within 254)
__global__ void dist_rows_kernel(const unsigned char *occ, unsigned char *d1, int nx, int ny) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= (long long)nx * ny) return;
    const int y = (int)(c / nx), x = (int)(c - (long long)y * nx);
    const unsigned char *row = occ + (long long)y * nx;
    int best = 255;
    for (int r = 0; r < best; r++)
        if ((x - r >= 0 && row[x - r]) || (x + r < nx && row[x + r])) { best = r; break; }
    d1[c] = (unsigned char)best;
}

// dist[y][x] = min over rows y' of max(|y - y'|, d1[y'][x])
__global__ void dist_cols_kernel(const unsigned char *d1, unsigned char *dist, int nx, int ny) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= (long long)nx * ny) return;
    const int y = (int)(c / nx);
    int best = d1[c];
    for (int r = 1; r < best; r++) {
        if (y - r >= 0) best = min(best, max(r, (int)d1[c - (long long)r * nx]));
        if (y + r < ny) best = min(best, max(r, (int)d1[c + (long long)r * nx]));
    }
    dist[c] = (unsigned char)best;
}

// mark: scratch of ncell ints; d1: scratch of ncell bytes; occ, dist: ncell bytes each; nempty: zeroed here
cudaError_t launch_build_distance_field(const float *chi, const float *eta, const float *line, const unsigned char *active, int nx, int ny,
                                        int L, int *mark, unsigned char *occ, unsigned char *d1, unsigned char *dist,
                                        unsigned long long *nempty, cudaStream_t st) {
    const long long ncell = (long long)nx * ny;
    cudaError_t e = cudaMemsetAsync(mark, 0, sizeof(int) * (size_t)ncell, st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(nempty, 0, sizeof(*nempty), st);
    if (e != cudaSuccess) return e;
    // a cell is empty when chi and eta vanish at every wavelength (emission without opacity counts, reading G11);
    // line mode: the six line parameters, of which chi_c and chi_line decide - S and v alone emit and absorb nothing
    const float *fields[2] = {line ? line : chi, line ? nullptr : eta};
    const int width = line ? 6 : L;
    for (const float *f : fields) {
        if (f == nullptr) continue;
        if (!line && width % 4 == 0 && (reinterpret_cast<uintptr_t>(f) & 15) == 0)
            mark_occupied_kernel<4><<<148 * 16, 256, 0, st>>>(f, ncell * (width / 4), width / 4, mark, 0xf);
        else
            mark_occupied_kernel<1><<<148 * 16, 256, 0, st>>>(f, ncell * width, width, mark, line ? 0x5 : 0xffffffffu);
    }
    const unsigned blocks = (unsigned)((ncell + 255) / 256);
    occupancy_kernel<<<blocks, 256, 0, st>>>(mark, active, occ, ncell, nempty);
    dist_rows_kernel<<<blocks, 256, 0, st>>>(occ, d1, nx, ny);
    dist_cols_kernel<<<blocks, 256, 0, st>>>(d1, dist, nx, ny);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Geometric work count: the number of (probe, direction) cell segments of one cascade that lie inside
// the box, per wavelength — the unit of BASELINE.json's metric: the sum over probes and directions of
// the in-box step counts march_kernel itself uses.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) count_kernel(MarchParams p, unsigned long long *total) {
    const int lane = threadIdx.x & 31;
    const long long W = (long long)blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5);
    if (W >= (p.qlist != nullptr ? (long long)(p.qpad >> 3) * (p.fix ? 4 : 1) : p.plist != nullptr ? (long long)p.npatch_act : (long long)p.npatch_x * p.npatch_y * (p.fix ? 4 : 1)) * p.ngroups || p.cnt == nullptr) return;
    const WarpWork ww = warp_work(p, W, lane);  // batch index is the slowest: W covers batch 0 only
    const int a = ww.a, b = ww.b, kg = ww.kg;
    const int s = 1 << p.shift, half = s >> 1;
    const int Y0 = (b << p.shift) + half;
    const int dxlo = -(a << p.shift) - half, dxhi = ((p.npx - a) << p.shift) - 1 - half;
    const int dylo = -Y0, dyhi = p.ny - 1 - Y0;
    unsigned long long mine = 0;
    for (int jj = 0; jj < (p.fix ? 16 : 4); jj++) {
        const long long tid = p.fix ? (4LL * kg + (jj >> 2)) * 16 + ww.cls * 4 + (jj & 3) : 4LL * kg + jj;
        const long long o = __ldg(p.off + tid);
        const int n = __ldg(p.cnt + tid);
        int nin = steps_inside(p.xy + o, n, ww.valid, dxlo, dxhi, dylo, dyhi);
        if (p.fix && n > 0) {
            const unsigned e = __ldg(reinterpret_cast<const unsigned *>(p.xy + o));
            const int dx = (int)(short)(e & 0xffffu), dy = (int)(short)(e >> 16);
            if (dx < dxlo || dx > dxhi || dy < dylo || dy > dyhi) nin = 0;
        }
        mine += (unsigned long long)nin;
    }
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_down_sync(FULL, mine, o);
    if (lane == 0 && mine) atomicAdd(total, mine);
}

cudaError_t launch_count(const MarchParams &p, unsigned long long *total, cudaStream_t st) {
    const long long nwarps = (p.qlist != nullptr ? (long long)(p.qpad >> 3) * (p.fix ? 4 : 1) : p.plist != nullptr ? (long long)p.npatch_act : (long long)p.npatch_x * p.npatch_y * (p.fix ? 4 : 1)) * p.ngroups;
    const long long blocks = (nwarps + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (blocks == 0) return cudaSuccess;
    count_kernel<<<(unsigned)blocks, WARPS_PER_BLOCK * 32, 0, st>>>(p, total);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Diagonal approximate lambda operator of cascade 0 (eq. 17): Lambda* = exp(-chi ds), ds from
// the cell centre to its edge along a cascade-0 ray = sqrt2/2 (diagonals), over sin(inclination) when inclined;
// mean over the 4 directions, summed over the inclinations with their weights.  One thread per (cell, wavelength).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) alo_kernel(AloParams p) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.ncell * p.L) return;
    const float HALF_DIAG = 0.70710678118654752f;
    float out = 0.f;
    if (p.line == nullptr) {
        const float c = __ldg(p.chi + i);
        for (int m = 0; m < p.nm; m++) out = fmaf(p.w[m], expf(-c * HALF_DIAG * p.f[m]), out);
    } else {
        const long long cell = i / p.L;
        const int l = (int)(i - cell * p.L);
        const float *q = p.line + cell * 6;
        const float chi_c = __ldg(q), chi_l = __ldg(q + 2), vx = __ldg(q + 4), vy = __ldg(q + 5), x = __ldg(p.xl + l);
        for (int m = 0; m < p.nm; m++) {
            float acc = 0.f;
            for (int k = 0; k < 4; k++) {  // the four diagonals; photons travel along -w: a = x_l + v.w sin(inclination)
                const float wx = (k == 0 || k == 3) ? HALF_DIAG : -HALF_DIAG, wy = k < 2 ? HALF_DIAG : -HALF_DIAG;
                const float a = x + (vx * wx + vy * wy) / p.f[m];
                const float c = fmaf(chi_l, expf(-a * a) * 0.5641895835477563f, chi_c);
                acc += expf(-c * HALF_DIAG * p.f[m]);
            }
            out = fmaf(p.w[m], 0.25f * acc, out);
        }
    }
    p.out[i] = out;
}

cudaError_t launch_alo(const AloParams &p, cudaStream_t st) {
    const long long n = p.ncell * p.L;
    alo_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Measurement aid (rc_probe_gather_bandwidth): the march's access pattern with nothing else — every
// warp reads pseudo-random 1 KB runs (32 lanes x 32 B, LDG.256), two in flight per warp, 48 warps per
// SM — over a region of `nsector` 32-byte sectors.  Region inside L2: the L2 -> SM gather ceiling.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned hash32(unsigned x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

__global__ void __launch_bounds__(256) gather_probe_kernel(const float *buf, unsigned long long nsector, int iters, float *sink) {
    const int lane = threadIdx.x & 31;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    float acc = 0.f;
    for (int it = 0; it < iters; it += 2) {
        float v[2][8];
#pragma unroll
        for (int u = 0; u < 2; u++) {
            // (a multiply-high, not a 64-bit modulo: with `%` the probe was bound by its own address arithmetic and read
            // 18.2 TB/s where the L2 -> SM path delivers 19.8-20.0, round 2)
            const unsigned long long c = __umulhi(hash32(warp * 7919u + it + u), (unsigned)(nsector - 32));
            load_vec<8>(buf + (c + lane) * 8, v[u]);
        }
#pragma unroll
        for (int u = 0; u < 2; u++)
#pragma unroll
            for (int k = 0; k < 8; k++) acc += v[u][k];
    }
    if (acc == 12345.678f) sink[0] = acc;  // never true in practice: keeps the loads alive
}

// The same pattern staged through shared memory with the TMA bulk-copy engine instead of LDG: every warp owns a
// ring of D = 4 stages x 2 KB, one lane issues two 1 KB `cp.async.bulk` copies per step (SASS: UBLKCP) that
// complete on an mbarrier, all lanes then read their 2 x 32 bytes with LDS.128.  This is the "TMA staging of
// the grid tile" design measured against the LDG path in DESIGN.md §7 (it is slower for 1 KB runs, so the
// march does not use it); kept as a probe so that the comparison can be repeated.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

template <int D, int WARPS>
__global__ void __launch_bounds__(WARPS * 32) bulk_probe_kernel(const float *buf, unsigned long long nsector, int iters, float *sink) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned char *ring = smem + (size_t)w * D * 2048;
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem + (size_t)WARPS * D * 2048) + w * D;
    if (lane == 0)
        for (int d = 0; d < D; d++) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bars + d)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncwarp();
    auto issue = [&](int it) {
        const unsigned bar = smem_u32(bars + it % D), dst = smem_u32(ring + (it % D) * 2048);
        const unsigned h = hash32(warp * 7919u + it);
        const float *s0 = buf + (h % (nsector - 64)) * 8, *s1 = buf + (hash32(h) % (nsector - 64)) * 8;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], 2048;" ::"r"(bar) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 1024, [%2];"
                     ::"r"(dst), "l"(s0), "r"(bar) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 1024, [%2];"
                     ::"r"(dst + 1024), "l"(s1), "r"(bar) : "memory");
    };
    if (lane == 0)
        for (int d = 0; d < D - 1 && d < iters; d++) issue(d);
    float acc = 0.f;
    for (int it = 0; it < iters; it++) {
        const unsigned bar = smem_u32(bars + it % D), parity = (it / D) & 1;
        asm volatile("{\n\t.reg .pred q;\n\tW_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 q, [%0], %1;\n\t@!q bra W_%=;\n\t}"
                     ::"r"(bar), "r"(parity) : "memory");
        const float4 *s4 = reinterpret_cast<const float4 *>(ring + (it % D) * 2048);
        const float4 a = s4[lane * 2], b = s4[lane * 2 + 1], c = s4[64 + lane * 2], d = s4[64 + lane * 2 + 1];
        __syncwarp();
        if (lane == 0 && it + D - 1 < iters) issue(it + D - 1);
        acc += a.x + a.y + a.z + a.w + b.x + b.y + b.z + b.w + c.x + c.y + c.z + c.w + d.x + d.y + d.z + d.w;
    }
    if (acc == 12345.678f) sink[0] = acc;
}

cudaError_t launch_bulk_probe(const float *buf, unsigned long long nsector, int iters, int sms, float *sink, cudaStream_t st, long long *bytes) {
    constexpr int D = 4, WARPS = 8;
    const size_t smem = (size_t)WARPS * D * 2048 + WARPS * D * 8;
    cudaError_t e = cudaFuncSetAttribute(bulk_probe_kernel<D, WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int blocks = sms * 3;  // 24 warps per SM, 192 KB of staging per SM
    bulk_probe_kernel<D, WARPS><<<blocks, WARPS * 32, smem, st>>>(buf, nsector, iters, sink);
    *bytes = (long long)blocks * WARPS * iters * 2048LL;
    return cudaGetLastError();
}

cudaError_t launch_gather_probe(const float *buf, unsigned long long nsector, int iters, int blocks, float *sink, cudaStream_t st) {
    gather_probe_kernel<<<blocks, 256, 0, st>>>(buf, nsector, iters, sink);
    return cudaGetLastError();
}

}  // namespace rc
