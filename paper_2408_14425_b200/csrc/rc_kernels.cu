// rc_kernels.cu — sm_100a kernels of the radiance-cascades hot path.
//
//   table_build_kernel  fp64 DDA of ONE ray per (cascade, direction), relative to the probe's lattice
//                       vertex.  All probes of a cascade sit at the same sub-cell position
//                       ((a+1/2) 2^i is an integer for i >= 1; a cell centre for i = 0),
//                       so every probe's ray in direction k is an integer translate of this one: the
//                       cells it crosses and the lengths inside them are shared.
//   pack_kernel         chi, eta [y][x][l]  ->  chi*log2(e), S = eta/chi in the probe-strided layout
//                       [batch][y][x mod s][x div s][LV]: the cells that 32 x-adjacent probes of
//                       cascade i touch at the same step are contiguous (coalesced gathers).
//   march_kernel        a1 (eq. 16 along the interval) + a2 (boundary)
//                       + a3 (bilinear parents, mean of the 4 children, merge eq. 11,
//                       PAPER.md:149-157, 199-207) + a4 on cascade 0 (J), fused.
//                       One warp = 32 adjacent probes x 1 direction group (4 child directions in
//                       turn) x LV wavelengths per lane; geometry is warp-uniform (no divergence from
//                       the DDA itself), radiance in fp32, I and T never leave registers.
#include "rc_internal.h"

#include <math_constants.h>

namespace rc {

static constexpr unsigned FULL = 0xffffffffu;
static constexpr int WARPS_PER_BLOCK = 8;

// ------------------------------------------------------------------------------------------------
// Geometry tables (fp64).  Restates PAPER.md:171-176 (shell [t_i, t_{i+1}]) and PAPER.md:314 (DDA).
// ------------------------------------------------------------------------------------------------
__global__ void table_build_kernel(TableBuildParams p) {
    long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= p.ndir) return;
    Step *out = p.steps + p.off[k];
    StepXY *oxy = p.xy + p.off[k];
    const long long cap = p.off[k + 1] - p.off[k];
    const int shift = p.cascade, s = 1 << shift, half = s >> 1, npx = p.nx >> shift;
    // cell (vertex + (dx, dy)) in the packed layout [y][x mod s][x div s], relative to the vertex's cell
    auto emit = [&](int n, int dx, int dy, double ds) {
        const int tx = dx + half;
        out[n].delta = dy * p.nx + (tx & (s - 1)) * npx + (tx >> shift) - half * npx;
        out[n].ds = (float)ds;
        oxy[n].dx = (int16_t)dx;
        oxy[n].dy = (int16_t)dy;
    };
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
    const long long blocks = (p.ndir + threads - 1) / threads;
    table_build_kernel<<<(unsigned)blocks, threads, 0, st>>>(p);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Pack: one thread per (batch, y, xm, xd); moves LV wavelengths of one cell.
// ------------------------------------------------------------------------------------------------
template <int LV>
__global__ void __launch_bounds__(256) pack_kernel(PackParams p) {
    const long long ncell = (long long)p.nx * p.ny;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= ncell * p.nb) return;
    const int nbI = (int)(idx / ncell);
    const long long c = idx - (long long)nbI * ncell;  // output cell index: (y*s + xm)*npx + xd
    const int npx = p.nx >> p.shift;
    const int y = (int)(c / p.nx);
    const int r = (int)(c - (long long)y * p.nx);
    const int xm = r / npx, xd = r - xm * npx;
    const int x = (xd << p.shift) + xm;
    const long long src = ((long long)y * p.nx + x) * p.L + (long long)nbI * LV;
    float c2[LV], S[LV];
#pragma unroll
    for (int v = 0; v < LV; v++) {
        const bool ok = nbI * LV + v < p.L;
        const float ch = ok ? __ldg(p.chi + src + v) : 0.f;
        const float et = ok ? __ldg(p.eta + src + v) : 0.f;
        c2[v] = ch * 1.4426950408889634f;           // tau in units of ln 2: T = 2^-tau2
        S[v] = ch > 0.f ? et / ch : 0.f;             // vacuum cells emit nothing (include/rc.h "Inputs")
    }
    float *oc = p.chiT + idx * LV, *os = p.ST + idx * LV;
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

cudaError_t launch_pack(const PackParams &p, int LV, cudaStream_t st) {
    const long long n = (long long)p.nx * p.ny * p.nb;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    switch (LV) {
        case 8: pack_kernel<8><<<blocks, 256, 0, st>>>(p); break;
        case 4: pack_kernel<4><<<blocks, 256, 0, st>>>(p); break;
        case 2: pack_kernel<2><<<blocks, 256, 0, st>>>(p); break;
        default: pack_kernel<1><<<blocks, 256, 0, st>>>(p); break;
    }
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

template <int LV>
__device__ __forceinline__ void load_vec(const float *p, float (&v)[LV]) {
    if constexpr (LV == 8) {
        // one 256-bit load (sm_100: LDG.E.256): 32 lanes x 32 B = 8 full 128-byte lines per request
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

// Position of child probe a among the n parents per axis: a/2 - 1/4 in parent index units, clamped
// at the lattice edge.  Weight `f` goes to q1.
__device__ __forceinline__ void parent_axis(int a, int n, int &q0, int &q1, float &f) {
    const int base = (a & 1) ? (a - 1) >> 1 : (a >> 1) - 1;
    f = (a & 1) ? 0.25f : 0.75f;
    q0 = min(max(base, 0), n - 1);
    q1 = min(max(base + 1, 0), n - 1);
}

// Warp -> work mapping shared by march_kernel and count_kernel.  A block holds G = min(ngroups, 8)
// ADJACENT direction groups of the same 32-probe chunk (their rays overlap near the probes: L1 reuse)
// and, when a cascade has fewer than 8 groups, 8/G neighbouring chunks.  Across blocks the probe
// chunk varies fastest, then the direction, then the wavelength batch: the blocks resident at any
// time share a narrow fan of directions (a few MB of step tables) and one batch's planes (L2).
struct WarpWork {
    int nbI, kg;
    long long pc;
    bool any;
};

__device__ __forceinline__ WarpWork warp_work(const MarchParams &p, long long npc) {
    const int w = threadIdx.x >> 5;
    const int G = min(p.ngroups, WARPS_PER_BLOCK), Pb = WARPS_PER_BLOCK / G;
    const long long pcb_n = (npc + Pb - 1) / Pb;
    const int kgb_n = p.ngroups / G;
    long long bid = blockIdx.x;
    const long long pcb = bid % pcb_n;
    bid /= pcb_n;
    const int kgb = (int)(bid % kgb_n);
    WarpWork r;
    r.nbI = (int)(bid / kgb_n);
    r.kg = kgb * G + (w % G);
    r.pc = pcb * Pb + (w / G);
    r.any = r.pc < npc && r.nbI < p.nb;
    return r;
}

__host__ __device__ inline long long march_blocks(int ngroups, long long npc, int nb) {
    const int G = ngroups < WARPS_PER_BLOCK ? ngroups : WARPS_PER_BLOCK, Pb = WARPS_PER_BLOCK / G;
    return ((npc + Pb - 1) / Pb) * (ngroups / G) * nb;
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

// One warp = 32 adjacent probes x 1 direction group (its 4 child directions in turn) x LV wavelengths
// per lane.  Per step the warp reads one 8-byte table entry (uniform address) and each lane its
// cell's LV opacities and source functions; the loads of step st+1 are in flight while step st is
// integrated, and the table is read two steps ahead.
template <int LV, int MINB>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32, MINB) march_kernel(MarchParams p) {
    const int lane = threadIdx.x & 31;
    const long long nprobe = (long long)p.npx * p.npy;
    const long long npc = (nprobe + 31) >> 5;
    const WarpWork ww = warp_work(p, npc);
    if (!ww.any) return;
    const int nbI = ww.nbI, kg = ww.kg;
    const long long probe = ww.pc * 32 + lane;
    const bool valid = probe < nprobe;
    const int b = valid ? (int)(probe / p.npx) : 0;
    const int a = valid ? (int)(probe - (long long)b * p.npx) : 0;
    const int s = 1 << p.shift, half = s >> 1;
    const int Y0 = (b << p.shift) + half;
    const long long ncell = (long long)p.nx * p.ny;
    const long long base = (long long)Y0 * p.nx + (long long)half * p.npx + a;  // the vertex's cell, packed layout
    const float *chi0 = p.chiT + ((long long)nbI * ncell + base) * LV;
    const float *S0 = p.ST + ((long long)nbI * ncell + base) * LV;
    const long long ndir = 4LL * p.ngroups;
    // (dx, dy) ranges that keep this lane's ray inside the box
    const int dxlo = -(a << p.shift) - half, dxhi = ((p.npx - a) << p.shift) - 1 - half;
    const int dylo = -Y0, dyhi = p.ny - 1 - Y0;

    float acc[LV];
#pragma unroll
    for (int v = 0; v < LV; v++) acc[v] = 0.f;

    for (int j = 0; j < 4; j++) {
        const long long k = 4LL * kg + j;
        float I[LV], tau[LV], T[LV];
#pragma unroll
        for (int v = 0; v < LV; v++) { I[v] = 0.f; tau[v] = 0.f; T[v] = 1.f; }
        // cnt == null: the whole cascade lies outside any box of this size (pure boundary term)
        if (p.cnt != nullptr) {
            const long long o = __ldg(p.off + k);
            const int n = __ldg(p.cnt + k);
            const uint2 *tab = reinterpret_cast<const uint2 *>(p.steps + o);
            const int nin = steps_inside(p.xy + o, n, valid, dxlo, dxhi, dylo, dyhi);
            const int nw = __reduce_max_sync(FULL, nin);  // steps this warp walks
            // a lane past its last in-box step re-reads its own vertex cell over ds = 0: no branch, no effect
            float c2[LV], S[LV], c2n[LV], Sn[LV];
            uint2 e0 = __ldg(tab), e1 = __ldg(tab + 1);  // slots have 4 spare entries at the end
            {
                const bool in = 0 < nin;
                const long long d = in ? (long long)(int)e0.x : 0;
                load_vec<LV>(chi0 + d * LV, c2);
                load_vec<LV>(S0 + d * LV, S);
            }
            float ds = 0 < nin ? __uint_as_float(e0.y) : 0.f;
            // a1: eq. 16 along the interval, front to back: with tau accumulated,
            // T_n = 2^-tau2_n and the cell's contribution is S (T_{n-1} - T_n)  [= S T (1 - e^{-chi ds})]
#pragma unroll 2
            for (int st = 0; st < nw; st++) {
                const bool inn = st + 1 < nin;
                const long long d = inn ? (long long)(int)e1.x : 0;
                load_vec<LV>(chi0 + d * LV, c2n);
                load_vec<LV>(S0 + d * LV, Sn);
                const float dsn = inn ? __uint_as_float(e1.y) : 0.f;
                e1 = __ldg(tab + st + 2);
#pragma unroll
                for (int v = 0; v < LV; v++) {
                    tau[v] = fmaf(c2[v], ds, tau[v]);
                    const float Tn = ex2_neg(tau[v]);
                    I[v] = fmaf(S[v], T[v] - Tn, I[v]);
                    T[v] = Tn;
                }
                if (p.early_exit && (st & 7) == 7) {
                    float tmin = tau[0];
#pragma unroll
                    for (int v = 1; v < LV; v++) tmin = fminf(tmin, tau[v]);
                    // every live lane opaque at every wavelength: T is exactly 0, nothing more can arrive
                    if (__all_sync(FULL, st >= nin || tmin > 126.f)) break;
                }
#pragma unroll
                for (int v = 0; v < LV; v++) { c2[v] = c2n[v]; S[v] = Sn[v]; }
                ds = dsn;
            }
        }
        if (p.Aup == nullptr) {
            // a2: boundary intensity enters on the top cascade only: rays heading up
            // (sin theta_k > 0  <=>  k < N/2) see I_above, rays heading down I_below
            const float *Ib = (2 * k < ndir) ? p.I_above : p.I_below;
#pragma unroll
            for (int v = 0; v < LV; v++) I[v] = fmaf(T[v], __ldg(Ib + nbI * LV + v), I[v]);
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
        for (int v = 0; v < LV; v++) acc[v] += I[v];
    }
    if (!valid) return;
#pragma unroll
    for (int v = 0; v < LV; v++) acc[v] *= 0.25f;  // mean over the 4 children (cascade 0: a4, J)
    if (p.mode == 0) {
        store_vec<LV>(p.out + (((long long)nbI * p.ngroups + kg) * nprobe + probe) * LV, acc);
    } else if (p.mode == 1) {
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

cudaError_t launch_march(const MarchParams &p, int LV, cudaStream_t st) {
    const long long nprobe = (long long)p.npx * p.npy;
    const long long blocks = march_blocks(p.ngroups, (nprobe + 31) >> 5, p.nb);
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const dim3 grid((unsigned)blocks), block(WARPS_PER_BLOCK * 32);
    // minimum resident blocks per SM (register cap) measured best on cfg 2: LV=8 -> 3 (80 regs), LV=4 -> 4 (64 regs)
    switch (LV) {
        case 8: march_kernel<8, 3><<<grid, block, 0, st>>>(p); break;
        case 4: march_kernel<4, 4><<<grid, block, 0, st>>>(p); break;
        case 2: march_kernel<2, 4><<<grid, block, 0, st>>>(p); break;
        default: march_kernel<1, 4><<<grid, block, 0, st>>>(p); break;
    }
    return cudaGetLastError();
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

// RC_VALIDATE: flag |= 1 if any chi/eta is negative or non-finite, |= 2 if eta > 0 where chi == 0.
__global__ void validate_kernel(const float *chi, const float *eta, long long n, int *flag) {
    int bad = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const float c = chi[i], e = eta[i];
        if (!(c >= 0.f) || !(e >= 0.f) || isinf(c) || isinf(e)) bad |= 1;
        if (c == 0.f && e > 0.f) bad |= 2;
    }
    if (bad) atomicOr(flag, bad);
}

cudaError_t launch_validate(const float *chi, const float *eta, long long n, int *flag, cudaStream_t st) {
    validate_kernel<<<148 * 8, 256, 0, st>>>(chi, eta, n, flag);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Geometric work count: the number of (probe, direction) cell segments of one cascade that lie inside
// the box, per wavelength — the unit of BASELINE.json's metric: the sum over probes and directions of
// the in-box step counts march_kernel itself uses.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) count_kernel(MarchParams p, unsigned long long *total) {
    const int lane = threadIdx.x & 31;
    const long long nprobe = (long long)p.npx * p.npy;
    const long long npc = (nprobe + 31) >> 5;
    const long long nwarps = npc * p.ngroups;
    const long long W = (long long)blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5);
    if (W >= nwarps || p.cnt == nullptr) return;
    const long long pc = W / p.ngroups;
    const int kg = (int)(W - pc * p.ngroups);
    const long long probe = pc * 32 + lane;
    const bool valid = probe < nprobe;
    const int b = valid ? (int)(probe / p.npx) : 0;
    const int a = valid ? (int)(probe - (long long)b * p.npx) : 0;
    const int s = 1 << p.shift, half = s >> 1;
    const int Y0 = (b << p.shift) + half;
    const int dxlo = -(a << p.shift) - half, dxhi = ((p.npx - a) << p.shift) - 1 - half;
    const int dylo = -Y0, dyhi = p.ny - 1 - Y0;
    unsigned long long mine = 0;
    for (int j = 0; j < 4; j++) {
        const long long k = 4LL * kg + j;
        const long long o = __ldg(p.off + k);
        mine += (unsigned long long)steps_inside(p.xy + o, __ldg(p.cnt + k), valid, dxlo, dxhi, dylo, dyhi);
    }
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_down_sync(FULL, mine, o);
    if (lane == 0 && mine) atomicAdd(total, mine);
}

cudaError_t launch_count(const MarchParams &p, unsigned long long *total, cudaStream_t st) {
    const long long nprobe = (long long)p.npx * p.npy;
    const long long nwarps = ((nprobe + 31) >> 5) * p.ngroups;
    const long long blocks = (nwarps + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    count_kernel<<<(unsigned)blocks, WARPS_PER_BLOCK * 32, 0, st>>>(p, total);
    return cudaGetLastError();
}

}  // namespace rc
