// rc_internal.h — shared between rc_api.cu (C ABI, host logic) and rc_kernels.cu (sm_100a kernels).
// Not part of the public interface (include/rc.h is).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rc {

// One step of a ray through the grid, shared by every probe of the cascade (they are integer
// translates of one another).  `delta` is the offset, in cells of the cascade's packed layout
// [y mod s][x mod s][y div s][x div s], from the probe's own entry (b, a) of phase plane 0 to the
// cell the ray is in; `ds` the path length inside it.  8 bytes, read warp-uniformly.
struct Step {
    int32_t delta;
    float ds;
};

// The same step as (dx, dy) cell offsets: only used to find, per probe, how many steps lie in the box.
struct StepXY {
    int16_t dx, dy;
};

// Per-cascade geometry tables (device memory, inside the workspace).
struct CascadeTable {
    const Step *steps;      // all directions back to back
    const long long *off;   // [N+1] start of direction k's slot in `steps` (host-computed bounds)
    const int *cnt;         // [N]   entries actually used by direction k (device-built)
    long long total_slots;  // sum of slot sizes
    int empty;              // every direction's interval lies outside any box of this size
};

struct MarchParams {
    const float *chiT;  // packed opacity * log2(e): [nb][s][s][npy][npx][LV]  (phase (y mod s, x mod s), then y div s, x div s)
    const float *ST;    // packed source function eta/chi, same layout
    const float *linepk;  // null, or line mode: packed line parameters [s][s][npy][npx][6] (pack_line_kernel)
    const float *xls;     // line mode: [Lpad] wavelengths x_l * sqrt(log2 e), device
    const unsigned char *dist;  // null (lock-step march), or [ny][nx] Chebyshev distance to the nearest occupied cell (0 = occupied):
                                // every lane walks its own ray and jumps over empty space; packed arrays in cell order (shift 0)
    int sparse_mode;            // launch variant of the distance-field march (rc_kernels.cu, launch_march_sparse)
    const unsigned *hit_off;    // null, or the hit lists of this cascade (rc_analyse_atmosphere): [4 nx ny + 1] offsets, ray = probe * N_i + k,
    const unsigned short *hit_list;  // and the step numbers of every ray's occupied in-box cells; the packed arrays are then cell-major
    int list_b;                 // wavelength batches per warp of the march over hit lists: 1, 2, 4 or 8
    unsigned long long *walked; // null, or a counter of the cell segments actually integrated (rc_count_walked; per wavelength batch)
    const unsigned char *flags; // null (every probe), or [npy][npx]: the flagged probes of this cascade
    const int *plist;           // null, or the numbers of the patches that hold a flagged probe (npatch_act of them)
    int npatch_act;
    // null, or [ngroups / 8][qpad]: for every block of 8 direction groups the quads (4 x-adjacent probes) of the lattice
    // ordered by the in-box length of their rays; a warp takes 8 consecutive entries (0xffff: none), so that its 32
    // lock-step lanes finish together (DESIGN.md §7 "lane utilisation")
    const unsigned short *qlist;
    int qpad;
    const float *Aup;   // merged cascade i+1, pre-averaged over the 4 children: [nb][N_i][npy/2][npx/2][LV]; null on the top cascade
    float *out;         // mode 0: A_i [nb][N_i/4][npy][npx][LV]; mode 1: J [ny][nx][L]; mode 2: Jpart [nb][ny][nx]
    const Step *steps;
    const StepXY *xy;
    const long long *off;
    const int *cnt;
    const float *I_below;  // [Lpad][NM] device (one value per channel)
    const float *I_above;  // [Lpad][NM] device
    const float *weights;  // [Lpad] device
    int nx, ny, L, nb;     // nb: wavelength batches this launch covers,
    int nb0;               // starting at batch nb0 (0 except for the two halves of rc_solve_J_host's pipeline)
    int cascade, shift;    // s = 1 << shift
    int npx, npy;          // probes per axis of this cascade
    int ngroups;           // direction groups = 4^cascade (4 directions each)
    int mode;
    int early_exit;
    float tau_cut;         // a warp stops once every live lane has tau log2(e) above this at all its channels (126: T == 0 exactly)
    int pw_log2;           // one warp's 32 probes form a patch 2^pw_log2 wide, 32 >> pw_log2 high
    int npatch_x, npatch_y;  // patches per axis
    int fix;               // bilinear fix: 4 sub-rays per ray, lanes = probes of one parity class,
                           // packed layout of spacing 2s, tables indexed (k*16 + class*4 + slot)
    const float2 *subdir;  // fix: unit direction of each sub-ray (line mode)
    int cpw;               // child-per-warp: the 4 child directions of a group in 4 neighbouring warps (8 warps per block)
    int kg_n, kg_off;      // the launch covers direction groups (kg_off + 0 .. kg_n-1) mod ngroups
    // banded launch (state != null): only the steps inside [band_lo, band_hi) along band_axis
    // (0 = rows, 1 = columns), for rays travelling in direction band_sign along that axis
    float *state;          // parked rays: [nb][ngroups][4][npy][npx][2][LV]  (I, tau*log2 e)
    int band_axis, band_sign, band_lo, band_hi, band_final;
    // 2.5D inclination quadrature: path scale 1/sqrt(1 - mu_m^2) and weight of inclination m
    float incl_f[8], incl_w[8], incl_s[8];  // incl_s = sqrt(1 - mu^2): projection of in-plane velocities (line mode)
};

struct PackParams {
    const float *chi, *eta;  // [ny][nx][L]
    float *chiT, *ST;        // [nb][s][s][npy][npx][LV]
    const unsigned char *active;  // null, or [ny][nx]: cells that are not flagged are packed as vacuum
    int nx, ny, L, nb, shift;
    int nb0;                 // first wavelength batch of this launch (nb of them)
    float c_thin;            // cells with chi log2e below this are packed in the thin form (seg_update*() in rc_kernels.cu)
    int list_b;              // > 0: write [batch group of list_b][cell][batch in group][LV] (march over hit lists, shift 0)
    // small grids (launch bound): nmulti > 0 packs for nmulti cascades in one launch, cascade j (blockIdx.y) with spacing
    // 2^shifts[j] into chiTm[j], STm[j]; shift, chiT, ST above are then unused
    int nmulti;
    int shifts[12];                    // (12 = RC_MAX_CASCADES of rc.h)
    float *chiTm[12], *STm[12];
};

struct AloParams {
    const float *chi;   // GivenFs: [ncell][L]; null in line mode
    const float *line;  // line mode: [ncell][6] as given by the caller; else null
    const float *xl;    // line mode: [L] wavelengths (Doppler widths, unscaled), device
    float *out;         // [ncell][L]
    long long ncell;
    int L, nm;
    float f[8], w[8];   // path scale and weight of each inclination
};

struct TableBuildParams {
    Step *steps;
    StepXY *xy;
    const long long *off;
    int *cnt;
    int cascade, top;
    long long ndir;
    double ta, tb;  // interval ends (tb = +inf on the top cascade)
    int nx, ny;
    int fix;         // bilinear fix: 16 tables per direction (parity class x parent slot), off/cnt indexed k*16 + sub
    float2 *subdir;  // fix: [ndir*16] unit direction of each sub-ray
};

// launchers (rc_kernels.cu); LV in {1,2,4,8}
cudaError_t launch_pack(const PackParams &p, int LV, cudaStream_t st);
cudaError_t launch_pack_line(const PackParams &p, cudaStream_t st);  // p.chi = line [ny][nx][6], p.chiT = packed [..][6]
cudaError_t launch_march(const MarchParams &p, int LV, int NM, int variant, cudaStream_t st);
cudaError_t launch_table_build(const TableBuildParams &p, cudaStream_t st);
cudaError_t launch_reduce_jbar(const float *Jpart, float *Jbar, long long ncell, int nb, cudaStream_t st);
cudaError_t launch_count(const MarchParams &p, unsigned long long *total, cudaStream_t st);
cudaError_t launch_gather_probe(const float *buf, unsigned long long nsector, int iters, int blocks, float *sink, cudaStream_t st);
cudaError_t launch_flags_from_active(const unsigned char *active, unsigned char *flag0, long long ncell, cudaStream_t st);
cudaError_t launch_count_flags(const unsigned char *a, long long n, unsigned long long *out, cudaStream_t st);
cudaError_t launch_flag_parents(const unsigned char *child, int npx, int npy, unsigned char *parent, cudaStream_t st);
cudaError_t launch_mark_and_compact_patches(const MarchParams &p, int npatch, unsigned char *mark, int *list, int *count, cudaStream_t st);
cudaError_t launch_build_distance_field(const float *chi, const float *eta, const float *line, const unsigned char *active, int nx, int ny,
                                        int L, int *mark, unsigned char *occ, unsigned char *d1, unsigned char *dist,
                                        unsigned long long *nempty, cudaStream_t st);
cudaError_t launch_alo(const AloParams &p, cudaStream_t st);
cudaError_t launch_hit_walk(const MarchParams &p, bool fill, unsigned *cnt_or_off, unsigned short *list, unsigned long long *total, cudaStream_t st);
cudaError_t launch_occ_differs(const unsigned char *a, const unsigned char *b, long long n, int *flag, cudaStream_t st);
cudaError_t launch_hit_scan(unsigned *a, long long n, unsigned *bsum, unsigned long long total, cudaStream_t st);
cudaError_t launch_bulk_probe(const float *buf, unsigned long long nsector, int iters, int sms, float *sink, cudaStream_t st, long long *bytes);
cudaError_t launch_validate(const float *chi, const float *eta, long long n, int *flag, cudaStream_t st);

}  // namespace rc
