// fdas_harmsum.cu -- incoherent harmonic summing and candidate compaction
// (BASELINE.json configs[4]; "pulse harmonics").
#include "fdas_common.cuh"
#include <math.h>

struct HarmThr { float t[5]; };

// One CTA per tile of HS_COLS = 128 plane columns x all n_z rows: warp w walks rows w, w+8, ...; a lane
// owns the HS_CPT (2 or 4) cells col0 + lane + 32 j of the row.  S_1 = P; stage 2H adds the odd-h terms of
// fraction h/(2H) (the rounding rule is invariant under (h,H)->(2h,2H), so S_2H = S_H + odd terms).
//   k_h = floor((k h + H/2)/H), zeta_h = sgn(zeta) floor((|zeta| h + H/2)/H)   (include/fdas.h)
// Index arithmetic is done once per lane and row: stepping k by 32 moves k_h by exactly 32 h/H (an
// integer for H <= 16), so the other three cells reuse the first cell's source address plus a
// compile-time offset.  The 15 stretched streams of a tile touch ~4.84 x the tile's cells, each
// needed by ~1/f^2 cells of the tile; keeping whole columns of the tile in one CTA lets the L1 serve
// that reuse.  The f = 1 stream is read once (streaming load).
// grid = ceil(n_cols/(32 HS_CPT)), block = (32, 8).
constexpr int HS_ROWS_PER_PASS = 8;

// out of line: rare (called by all 32 lanes of a warp, see push_cand_warp)
__device__ __noinline__ void push_cand_hs(fdas_cand* list, uint32_t* count, uint32_t cap, bool hit,
                                          int col, int zi, int nharm, float power)
{
    push_cand_warp(list, count, cap, hit, col, zi, nharm, power);
}

// CHECK = true: edge tiles (first tile: k_h may fall below bin0; last tile: columns beyond n_cols).
//
// A warp takes a run of CONSECUTIVE rows of the tile (one lane = HS_CPT cells, columns col0 + 32 j).  For
// stream h/H the source column k_h does not depend on the row, and the source row zeta_h is non-decreasing
// in zeta and repeats over ~H/h consecutive rows.  So each stream keeps one pointer per thread that is
// advanced by one plane row when zeta_h moves, and a stream whose zeta_h did not move keeps last row's
// values: (16 + 8.5 (R-1))/R loads per cell for a run of R rows instead of 16, and no per-row index
// arithmetic.  Whether zeta_h moved is the same for the whole warp; lane s works it out for slot s
// (h, H of that slot) and one ballot hands the 16-bit answer to everybody:
//   t = |zeta| h + H/2, zeta_h = sgn(zeta) (t >> log2 H); against the previous row (|zeta| - 1 for
//   zeta > 0, |zeta| + 1 for zeta <= 0) it moved iff (t mod H) < h, resp. (t mod H) + h >= H.
// Stage st (H = 2^st) occupies slots [H/2, H): slot = H/2 + (h - 1)/2 for odd h; slot 0 is P itself.
template <int NST, int HS_CPT, bool CHECK>
__device__ __forceinline__ void harmsum_tile(const float* __restrict__ plane, fdas_cand* __restrict__ cands,
                                             uint32_t* __restrict__ count, uint32_t cap, const HarmThr& thr,
                                             int n_cols, int n_z, int bin0, int tile, int zi_lo, int zi_hi,
                                             int row_part, int n_row_parts)
{
    constexpr int HS_COLS = 32 * HS_CPT;
    constexpr int HMAX = 1 << (NST - 1);
    const int lane = threadIdx.x;
    const int col0 = tile * HS_COLS + lane;
    const int zc = (n_z - 1) / 2;
    const int k = bin0 + col0;
    const int rpw = (zi_hi - zi_lo + n_row_parts - 1) / n_row_parts;
    const int r_begin = zi_lo + row_part * rpw, r_end = min(zi_hi, r_begin + rpw);
    if (r_begin >= r_end) return;                                      // the whole warp

    // this lane's slot for the ballot (lanes 0 and >= HMAX never report a move)
    int my_h = 0, my_H = 1;
    if (lane >= 1 && lane < HMAX) {
        my_H = 2 << (31 - __clz(lane));
        my_h = 2 * (lane - (my_H >> 1)) + 1;
    }
    // one plane index per stream (n_z n_cols < 2^31, checked by the launcher), set ONE ROW BEFORE the first
    // source row: the first row moves every stream
    int idx[HMAX];
    unsigned long long okmask = 0;                                     // CHECK only: bit slot*HS_CPT + j = cell may be read
    {
        const int zeta0 = r_begin - zc, az0 = abs(zeta0), sg0 = zeta0 < 0 ? -1 : 1;
        idx[0] = r_begin * n_cols + col0;
#pragma unroll
        for (int j = 0; j < HS_CPT; j++)
            if (col0 + 32 * j < n_cols) okmask |= 1ull << j;
#pragma unroll
        for (int st = 1; st < NST; st++) {
            const int H = 1 << st;
#pragma unroll
            for (int h = 1; h < H; h += 2) {
                const int slot = (H >> 1) + (h >> 1);
                const int kh = (k * h + (H >> 1)) >> st;              // k*h < 2^29 for n_samples <= 2^25
                const int zh0 = sg0 * ((az0 * h + (H >> 1)) >> st);
                idx[slot] = (zc + zh0 - 1) * n_cols + (kh - bin0);
                if (CHECK) {
#pragma unroll
                    for (int j = 0; j < HS_CPT; j++)
                        if (kh + ((32 * h) >> st) * j >= bin0 && col0 + 32 * j < n_cols) okmask |= 1ull << (slot * HS_CPT + j);
                }
            }
        }
    }
    static_assert(HS_CPT % 2 == 0, "cells are summed in pairs (packed f32x2 adds)");
    // the row stride in a register of its own: otherwise every predicated index update re-reads it from the
    // constant bank (an LDC per stream and row)
    // (ptxas re-materialises a plain copy of a kernel parameter; gridDim.y is 1, which it cannot know)
    const int stride = n_cols + (int)gridDim.y - 1;
    float2 v[HS_CPT / 2][HMAX];                                       // .x, .y = cells 2jj, 2jj+1 of the lane
#define HS_V(j, i) (((j) & 1) ? v[(j) >> 1][i].y : v[(j) >> 1][i].x)
    for (int zi = r_begin; zi < r_end; zi++) {
        const int zeta = zi - zc;
        const int t = abs(zeta) * my_h + (my_H >> 1), fr = t & (my_H - 1);
        unsigned moved = __ballot_sync(0xffffffffu, zeta > 0 ? fr < my_h : fr + my_h >= my_H);
        if (zi == r_begin) moved = 0xffffffffu;
        // issue every gather of the row first (all independent), then sum in stage order
        {
            const float* src = plane + idx[0];
#pragma unroll
            for (int j = 0; j < HS_CPT; j++) HS_V(j, 0) = (!CHECK || (okmask >> j & 1)) ? __ldcs(src + 32 * j) : 0.0f;
            idx[0] += stride;
        }
#pragma unroll
        for (int st = 1; st < NST; st++) {
            const int H = 1 << st;
#pragma unroll
            for (int h = 1; h < H; h += 2) {
                const int slot = (H >> 1) + (h >> 1);
                if (moved & (1u << slot)) {                            // warp-uniform
                    idx[slot] += stride;
                    const float* src = plane + idx[slot];
                    const int dk = (32 * h) >> st;                     // exact: 32 h / H
#pragma unroll
                    for (int j = 0; j < HS_CPT; j++)
                        HS_V(j, slot) = (!CHECK || (okmask >> (slot * HS_CPT + j) & 1)) ? __ldg(src + dk * j) : 0.0f;
                }
            }
        }
#pragma unroll
        for (int jj = 0; jj < HS_CPT / 2; jj++) {
            // the stage sums of two cells at a time (FADD2: one issue slot for both), and ONE branch for the
            // (rare) cell that passes any threshold
            float2 sum[NST];
            float2 acc = v[jj][0];
            sum[0] = acc;
            bool any = acc.x > thr.t[0] || acc.y > thr.t[0];
#pragma unroll
            for (int st = 1; st < NST; st++) {
                const int H = 1 << st;
#pragma unroll
                for (int i = H >> 1; i < H; i++) acc = __fadd2_rn(acc, v[jj][i]);
                sum[st] = acc;
                any = any || acc.x > thr.t[st] || acc.y > thr.t[st];
            }
            if (__any_sync(0xffffffffu, any)) {                         // warp-uniform: the ballots below see all 32 lanes
#pragma unroll
                for (int st = 0; st < NST; st++) {
                    push_cand_hs(cands, count, cap, sum[st].x > thr.t[st] && (!CHECK || (okmask >> (2 * jj) & 1)),
                                 col0 + 32 * (2 * jj), zi, 1 << st, sum[st].x);
                    push_cand_hs(cands, count, cap, sum[st].y > thr.t[st] && (!CHECK || (okmask >> (2 * jj + 1) & 1)),
                                 col0 + 32 * (2 * jj + 1), zi, 1 << st, sum[st].y);
                }
            }
        }
    }
#undef HS_V
}

// ---- interior tiles: the row body specialised on its move pattern --------------------------------------------
// Which streams move to a new source row depends only on |zeta| mod 16 and on the side of zeta = 0 (the
// condition above involves t mod H, H | 16): 32 patterns.  harmsum_tile evaluates the pattern at run time
// (ballot + R2P) and ptxas if-converts every stream into ~8 predicated instructions that issue whether or not
// the stream moved (129 instructions per row and 2 cells).  Here the pattern is a TEMPLATE argument: a row
// jumps (one warp-uniform switch) to the body compiled for its pattern, which contains exactly the pointer
// bumps and loads of the streams that move -- 8 of 15 on average -- into the registers that carry the values
// from row to row; no predicates, no index arithmetic (one 64-bit pointer per stream, bumped by the row
// stride), no ballot.  With 4 cells per lane the stage sums are 30 FADD2 and 20 compares per row.
__host__ __device__ constexpr unsigned hs_moved_mask(int r16, bool positive, int nst)
{
    unsigned m = 1u;                                                   // slot 0 (P itself) always moves
    for (int st = 1; st < nst; st++) {
        const int H = 1 << st;
        for (int h = 1; h < H; h += 2) {
            const int fr = (r16 * h + (H >> 1)) & (H - 1);
            if (positive ? fr < h : fr + h >= H) m |= 1u << ((H >> 1) + (h >> 1));
        }
    }
    return m;
}

template <int NST, int HS_CPT, unsigned MASK>
__device__ __forceinline__ void hs_fetch_row(const float* (&ptr)[1 << (NST - 1)], float2 (&v)[HS_CPT / 2][1 << (NST - 1)],
                                             long long stride)
{
#define HS_V(j, i) (((j) & 1) ? v[(j) >> 1][i].y : v[(j) >> 1][i].x)
    ptr[0] += stride;
#pragma unroll
    for (int j = 0; j < HS_CPT; j++) HS_V(j, 0) = __ldcs(ptr[0] + 32 * j);
#pragma unroll
    for (int st = 1; st < NST; st++) {
        const int H = 1 << st;
#pragma unroll
        for (int h = 1; h < H; h += 2) {
            const int slot = (H >> 1) + (h >> 1);
            if (MASK & (1u << slot)) {                                 // compile time
                ptr[slot] += stride;
                const int dk = (32 * h) >> st;                         // exact: 32 h / H
#pragma unroll
                for (int j = 0; j < HS_CPT; j++) HS_V(j, slot) = __ldg(ptr[slot] + dk * j);
            }
        }
    }
#undef HS_V
}

#define HS_CASE(R, POS) case R: hs_fetch_row<NST, HS_CPT, hs_moved_mask(R, POS, NST)>(ptr, v, stride); break;
#define HS_CASES(POS) HS_CASE(0, POS) HS_CASE(1, POS) HS_CASE(2, POS) HS_CASE(3, POS) HS_CASE(4, POS) HS_CASE(5, POS) HS_CASE(6, POS) \
    HS_CASE(7, POS) HS_CASE(8, POS) HS_CASE(9, POS) HS_CASE(10, POS) HS_CASE(11, POS) HS_CASE(12, POS) HS_CASE(13, POS)               \
    HS_CASE(14, POS) HS_CASE(15, POS)

// Interior tile (every k_h >= bin0, every column < n_cols): rows [zi_lo, zi_hi) of 32 HS_CPT columns, one warp.
template <int NST, int HS_CPT>
__device__ __forceinline__ void harmsum_tile_fast(const float* __restrict__ plane, fdas_cand* __restrict__ cands,
                                                  uint32_t* __restrict__ count, uint32_t cap, const HarmThr& thr,
                                                  int n_cols, int n_z, int bin0, int tile, int zi_lo, int zi_hi)
{
    constexpr int HS_COLS = 32 * HS_CPT;
    constexpr int HMAX = 1 << (NST - 1);
    static_assert(HS_CPT % 2 == 0, "cells are summed in pairs (packed f32x2 adds)");
    const int lane = threadIdx.x;
    const int col0 = tile * HS_COLS + lane;
    const int zc = (n_z - 1) / 2;
    const int k = bin0 + col0;
    if (zi_lo >= zi_hi) return;                                        // the whole warp
    const long long stride = n_cols;
    // one pointer per stream, ONE ROW BEFORE its first source row: the first row moves every stream
    const float* ptr[HMAX];
    {
        const int zeta0 = zi_lo - zc, az0 = abs(zeta0), sg0 = zeta0 < 0 ? -1 : 1;
        ptr[0] = plane + ((long long)(zi_lo - 1) * n_cols + col0);
#pragma unroll
        for (int st = 1; st < NST; st++) {
            const int H = 1 << st;
#pragma unroll
            for (int h = 1; h < H; h += 2) {
                const int slot = (H >> 1) + (h >> 1);
                const int kh = (k * h + (H >> 1)) >> st;              // k*h < 2^29 for n_samples <= 2^25
                const int zh0 = sg0 * ((az0 * h + (H >> 1)) >> st);
                ptr[slot] = plane + ((long long)(zc + zh0 - 1) * n_cols + (kh - bin0));
            }
        }
    }
    float2 v[HS_CPT / 2][HMAX];                                       // .x, .y = cells 2jj, 2jj+1 of the lane
#pragma unroll 1
    for (int zi = zi_lo; zi < zi_hi; zi++) {
        const int zeta = zi - zc, r16 = abs(zeta) & 15;                // warp-uniform
        if (zi == zi_lo) hs_fetch_row<NST, HS_CPT, 0xffffffffu>(ptr, v, stride);
        else if (zeta > 0) { switch (r16) { HS_CASES(true) } }
        else { switch (r16) { HS_CASES(false) } }
#pragma unroll
        for (int jj = 0; jj < HS_CPT / 2; jj++) {
            float2 sum[NST];
            float2 acc = v[jj][0];
            sum[0] = acc;
            bool any = acc.x > thr.t[0] || acc.y > thr.t[0];
#pragma unroll
            for (int st = 1; st < NST; st++) {
                const int H = 1 << st;
#pragma unroll
                for (int i = H >> 1; i < H; i++) acc = __fadd2_rn(acc, v[jj][i]);
                sum[st] = acc;
                any = any || acc.x > thr.t[st] || acc.y > thr.t[st];
            }
            if (__any_sync(0xffffffffu, any)) {                         // rare; warp-uniform: the ballots below see all 32 lanes
#pragma unroll
                for (int st = 0; st < NST; st++) {
                    push_cand_hs(cands, count, cap, sum[st].x > thr.t[st], col0 + 32 * (2 * jj), zi, 1 << st, sum[st].x);
                    push_cand_hs(cands, count, cap, sum[st].y > thr.t[st], col0 + 32 * (2 * jj + 1), zi, 1 << st, sum[st].y);
                }
            }
        }
    }
}
#undef HS_CASES
#undef HS_CASE

// Tile order.  The stretch (k, zeta) -> (k h/H, zeta h/H) moves a cell along the ray through the origin of
// the (k, zeta) plane, so the 16 cells that read one source cell all lie on that ray, at k = x H/h: with the
// plain order (all rows of a column tile together, columns ascending) they are 1/16 ... 15/16 of the plane
// apart in time and nothing is left in L2 (7.4 GB of DRAM reads for a 1.43 GB plane in an ncu capture; an LRU
// model of this order gives 7.36 GB).  The plane is therefore cut into S angular SECTORS of equal area that
// are swept one after the other, columns ascending inside each.  Boundary ray j = 0..S is named by where it
// leaves the rectangle [0, K] x [-n_z/2, n_z/2], u_j = -2 + 4 j/S:  |u| <= 1: through the far edge k = K at
// row (n_z/2) u;  1 < |u| <= 2: through the top/bottom edge at column K (2 - |u|)  (|u| = 2: vertical).
// Sector s holds, in the column tile whose last bin is kc, the rows ceil(zb_s(kc)) <= zeta < ceil(zb_{s+1}(kc))
// -- a partition of the rows of every tile.  A sector is thin, so the span of plane that streams through L2
// between two uses of a source cell fits (the same model: 1.54 GB at S = 16, 1.43-1.51 GB at S = 32 for a
// 90-60 MB cache: the plane is read from DRAM about once).  S = 1 is the plain order; results do not depend on S.
// The kernel is PERSISTENT: the grid holds as many CTAs as are resident at once and CTA c takes the work
// items c, c + gridDim.x, ... (item = one 32 HS_CPT-column tile of one sector, sector-major, columns
// ascending).  So the CTAs running at any moment work on ~gridDim.x consecutive tiles (~76 k columns of one
// sector) and advance together, which is what the reuse argument needs; one CTA per run of tiles would spread
// the resident CTAs over a quarter of the plane.
constexpr int HS_MAX_SECTORS = 64;
struct HarmSectors {
    int n_sec;
    int col_warps;                           // > 1: the warps of a CTA take ADJACENT column tiles (all rows each) and share
                                             // the L1 lines at the seams; 1: they split the rows of one tile (plain order)
    int first_item[HS_MAX_SECTORS + 1];      // sector s owns items [first_item[s], first_item[s+1]): its groups of col_warps tiles
};

__host__ __device__ inline double sector_boundary(int j, int S, double kc, double K, double zhalf)
{
    const double u = -2.0 + 4.0 * (double)j / (double)S, au = u < 0.0 ? -u : u;
    if (au <= 1.0) return zhalf * u * kc / K;
    const double c = K * (2.0 - au);
    const double r = (c <= 0.0 || kc >= c) ? 1.0 : kc / c;
    return u < 0.0 ? -zhalf * r : zhalf * r;
}

template <int NST, int HS_CPT, int MINB>
__global__ void __launch_bounds__(MINB >= 3 ? 128 : 256, MINB)           // MINB >= 3: at most 4 warps per CTA (the launcher sees to it)
k_harmsum(const float* __restrict__ plane, fdas_cand* __restrict__ cands, uint32_t* __restrict__ count,
          uint32_t cap, HarmThr thr, HarmSectors sec, int n_cols, int n_z, int bin0)
{
    constexpr int HS_COLS = 32 * HS_CPT;
    const int zc = (n_z - 1) / 2;
    const double K = (double)(bin0 + n_cols - 1), zhalf = 0.5 * (double)n_z;
    const int n_items = sec.first_item[sec.n_sec];
    const int n_tiles = (n_cols + HS_COLS - 1) / HS_COLS;
    int s = 0;
#pragma unroll 1
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {                // everything here is CTA-uniform
        while (item >= sec.first_item[s + 1]) s++;
        const int group = item - sec.first_item[s];
        const int tile_last = min(n_tiles, (group + 1) * sec.col_warps) - 1;
        int zi_lo = 0, zi_hi = n_z;
        if (sec.n_sec > 1) {                 // rows of this sector, taken at the last bin of the group of tiles
            const double kc = (double)bin0 + (double)min(n_cols, (tile_last + 1) * HS_COLS) - 1.0;
            zi_lo = max(0, min(n_z, (int)ceil(sector_boundary(s, sec.n_sec, kc, K, zhalf)) + zc));
            zi_hi = max(0, min(n_z, (int)ceil(sector_boundary(s + 1, sec.n_sec, kc, K, zhalf)) + zc));
            if (zi_lo >= zi_hi) continue;
        }
        const int tile = sec.col_warps > 1 ? group * sec.col_warps + (int)threadIdx.y : group;       // warp-uniform
        if (tile >= n_tiles) continue;
        const int row_part = sec.col_warps > 1 ? 0 : (int)threadIdx.y, n_row_parts = sec.col_warps > 1 ? 1 : (int)blockDim.y;
        const bool edge = tile == 0 || tile * HS_COLS + HS_COLS > n_cols;
        if (edge) {
            harmsum_tile<NST, HS_CPT, true>(plane, cands, count, cap, thr, n_cols, n_z, bin0, tile, zi_lo, zi_hi, row_part, n_row_parts);
        } else {                             // interior: this warp's rows of the tile (all of them, or its part in the plain order)
            const int rpw = (zi_hi - zi_lo + n_row_parts - 1) / n_row_parts;
            const int r_begin = zi_lo + row_part * rpw, r_end = min(zi_hi, r_begin + rpw);
            harmsum_tile_fast<NST, HS_CPT>(plane, cands, count, cap, thr, n_cols, n_z, bin0, tile, r_begin, r_end);
        }
    }
}

// Sector -> item ranges.  A sector whose two boundary rays both leave through the top/bottom edge is empty
// beyond the column where the shallower one leaves; only the tiles before that become items.
static HarmSectors make_sectors(int n_sec, int col_warps, int n_cols, int bin0, int cols_per_tile)
{
    HarmSectors hs;
    hs.n_sec = n_sec;
    hs.col_warps = col_warps;
    const int n_tiles = (n_cols + cols_per_tile - 1) / cols_per_tile;
    const double K = (double)(bin0 + n_cols - 1);
    hs.first_item[0] = 0;
    for (int s = 0; s < n_sec; s++) {
        int nt = n_tiles;
        if (n_sec > 1) {
            const double ua = -2.0 + 4.0 * s / n_sec, ub = -2.0 + 4.0 * (s + 1) / n_sec;
            const double umin = fabs(ua) < fabs(ub) ? fabs(ua) : fabs(ub);
            if (ua * ub > 0.0 && umin > 1.0) {
                const long long t = ((long long)(K * (2.0 - umin) / (cols_per_tile * col_warps)) + 2) * col_warps;
                if (t < nt) nt = (int)t;
            }
        }
        hs.first_item[s + 1] = hs.first_item[s] + (nt + col_warps - 1) / col_warps;
    }
    return hs;
}

// CTAs resident at once for kernel `k` with `threads` per CTA (the persistent grid).
template <class K>
static int resident_ctas(K k, int threads)
{
    int dev = 0, sms = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, threads, 0) != cudaSuccess || sms < 1 || per_sm < 1) {
        cudaGetLastError();
        return 148 * 4;
    }
    return sms * per_sm;
}

// Threshold + warp-ballot compaction over one plane (row a8): a thread tests 4 adjacent columns of a row (one
// 16-byte load where the address allows it -- the plane pointer itself need only be 4-byte aligned,
// include/fdas.h -- else scalar loads); each of the 4 is appended with one ballot and one atomic per warp.
// No thread leaves early: the ballots need the whole warp.   grid = (ceil(n_cols/1024), n_z), block 256.
__global__ void __launch_bounds__(256)
k_candidates(const float* __restrict__ plane, fdas_cand* __restrict__ cands, uint32_t* __restrict__ count,
             uint32_t cap, float thr, int n_cols)
{
    const int zi = blockIdx.y;
    const float* row = plane + (size_t)zi * n_cols;
    const int c4 = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
    float v[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    if (c4 + 3 < n_cols && (reinterpret_cast<uintptr_t>(row + c4) & 15) == 0) {
        const float4 q = __ldg(reinterpret_cast<const float4*>(row + c4));
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; i++)
            if (c4 + i < n_cols) v[i] = __ldg(row + c4 + i);
    }
#pragma unroll
    for (int i = 0; i < 4; i++)
        push_cand_warp(cands, count, cap, c4 + i < n_cols && v[i] > thr, c4 + i, zi, 1, v[i]);
}

int fdas_launch_harmsum(fdas_plan* p, const float* d_plane, int max_harm, const float* h_thr,
                        fdas_cand* d_cands, uint32_t* d_count, uint32_t cap, cudaStream_t st)
{
    if ((long long)p->n_z * p->n_cols > 0x7fffffffLL) return FDAS_E_INVALID;          // 32-bit plane indices in the kernel
    int n_stage = 0;
    for (int H = 1; H <= max_harm; H <<= 1) n_stage++;
    HarmThr thr;
    for (int i = 0; i < 5; i++) thr.t[i] = i < n_stage ? h_thr[i] : 3.0e38f;
    FDAS_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint32_t), st));
    int n_cols = (int)p->n_cols;
    const int variant = p->tune_hs_variant;
    // sectors of the tile order (see k_harmsum): 16 by default, thin enough for the reuse distance to fit in
    // L2, thick enough (~10 rows at the far end) for L1 to keep serving the row-direction reuse inside a stream
    const int env_sectors = p->tune_hs_sectors > 0 ? p->tune_hs_sectors : 16;
    const int env_rows = p->tune_hs_rows;
    int n_sec = env_sectors < 1 ? 1 : env_sectors;
    if (n_sec > HS_MAX_SECTORS) n_sec = HS_MAX_SECTORS;
    int rows = env_rows > 0 ? env_rows : (n_sec == 1 ? HS_ROWS_PER_PASS : 4);      // warps per CTA: with sectors, 4 adjacent column tiles (all rows of the
                                                                                    // sector each: longest carried runs); plain order: 8 row parts of one tile
    if (rows > HS_ROWS_PER_PASS) rows = HS_ROWS_PER_PASS;
    dim3 block(32, rows);
    HarmSectors sec;
#define FDAS_HS_LAUNCH(NST, CPT, MINB)                                                              \
    do {                                                                                            \
        if (MINB >= 3 && rows > 4) { rows = 4; block = dim3(32, rows); }   /* launch bound of that instance */ \
        sec = make_sectors(n_sec, n_sec == 1 ? 1 : rows, n_cols, p->bin0, 32 * CPT);                                       \
        int n_cta = resident_ctas(k_harmsum<NST, CPT, MINB>, 32 * rows);                            \
        if (n_cta > sec.first_item[n_sec]) n_cta = sec.first_item[n_sec];                           \
        k_harmsum<NST, CPT, MINB><<<dim3(n_cta), block, 0, st>>>(                                   \
            d_plane, d_cands, d_count, cap, thr, sec, n_cols, p->n_z, p->bin0);                     \
    } while (0)
    switch (n_stage) {
    case 1: FDAS_HS_LAUNCH(1, 4, 2); break;
    case 2: FDAS_HS_LAUNCH(2, 4, 2); break;
    case 3: FDAS_HS_LAUNCH(3, 4, 2); break;
    case 4: FDAS_HS_LAUNCH(4, 2, 2); break;
    default:
        if (variant == 1) FDAS_HS_LAUNCH(5, 2, 2);        // 64-column tiles, 128 registers, 4 CTAs/SM: ~45 instructions per cell (tuning key)
        else FDAS_HS_LAUNCH(5, 4, 3);                    // 128-column tiles, 3 CTAs of 4 warps per SM: ~33 instructions per cell (profiles/)
        break;
    }
#undef FDAS_HS_LAUNCH
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}

int fdas_launch_candidates(fdas_plan* p, const float* d_plane, float thr, fdas_cand* d_cands,
                           uint32_t* d_count, uint32_t cap, cudaStream_t st)
{
    FDAS_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint32_t), st));
    int n_cols = (int)p->n_cols;
    k_candidates<<<dim3((n_cols + 1023) / 1024, p->n_z), 256, 0, st>>>(d_plane, d_cands, d_count, cap, thr, n_cols);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}

int fdas_occupancy_harmsum(int32_t* ctas, int32_t* regs, int32_t* smem)
{
    return fdas_occupancy_of(k_harmsum<5, 4, 3>, 128, 0, ctas, regs, smem);
}
