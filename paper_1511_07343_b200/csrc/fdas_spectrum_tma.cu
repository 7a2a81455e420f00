// fdas_spectrum_tma.cu -- PAPER.md:49 step 2 for series of 2^13 samples and more: the real-to-complex FFT as a
// MULTI-PASS, TMA-STAGED transform (BASELINE.json north_star), plus the mean-power normalisation of
// BASELINE.json configs[0].  Shorter series take the generic kernels of fdas_spectrum.cu.
//
// The N real samples are packed as M = N/2 complex values z[n] = x[2n] + i x[2n+1]; M = Ra Rb Rc (three passes,
// M >= 2^17) or Ra Rc (two passes, Rb = 1), every factor in {32, 64, 128, 256}.  With
//   n = n_a Rb Rc + n_b Rc + n_c ,   k = k_a + Ra k_b + Ra Rb k_c     (W_n = exp(-2 pi i / n))
//   Z[k] = sum_nc W_Rc^{nc kc} W_M^{nc (ka + Ra kb)}  sum_nb W_Rb^{nb kb} W_{RaRb}^{nb ka}  sum_na W_Ra^{na ka} z[n]
// pass A  transforms n_a (the slowest index: rows of a [Ra][Rb Rc] matrix) and applies W_{RaRb}^{nb ka};
// pass B  transforms n_b for every k_a and applies W_M^{nc (ka + Ra kb)}; it writes row kappa = ka + Ra kb of a
//         [Ra Rb][Rc] matrix, so that the rows of the last pass are in natural frequency order;
// pass C  transforms the contiguous n_c of rows kappa and NR - kappa together (NR = Ra Rb rows), untangles the
//         real-input spectrum F_k = E_k + W_N^k O_k from Z_k and Z_{M-k}, scales by 1/sqrt(mu) and stores bins 1..N/2.
// A tile is always 4096 complex values (32 KB) worked on by 256 threads holding 16 values each: a transform of
// length R is a 16-point DFT in registers, a twiddle, ONE exchange through shared memory and R/16-point DFTs in
// registers.  Passes A and B ("column" passes: the transformed index is strided, 16..128 contiguous columns ride
// along) fetch their tile with one tensor-map box load and write it back with one box store; pass C ("row" pass)
// fetches its 16..128 rows with one bulk copy each.  Intermediates live in the output buffer and the workspace
// (33.5 MB each at 2^23 samples: L2-resident), so only the series read and the spectrum write reach HBM.
// mu = mean_{k=1..N/2} |F_k|^2 comes from the time domain by Parseval (reading R3): pass A accumulates
// sum x, sum x^2 and sum (-1)^n x in fp64 per tile, k_spec_scale reduces them in a fixed order.
#include "fdas_common.cuh"
#include "fdas_regfft.cuh"
#include "fdas_tma.cuh"
#include <string.h>

constexpr int SPT_THREADS = 256;
constexpr int SPT_TILE = 4096;                       // complex values per tile
constexpr int SPT_TILE_BYTES = SPT_TILE * 8;

// bit reversal of a `bits`-bit index (compile time after unrolling)
__host__ __device__ constexpr int brev(int j, int bits)
{
    int r = 0;
    for (int b = 0; b < bits; b++) r |= ((j >> b) & 1) << (bits - 1 - b);
    return r;
}

// forward DFT of R = 2^LR points (R <= 16) held in v[0..R) in NATURAL order, result in natural order.
// (the radix-2 stages of fdas_regfft.cuh want bit-reversed input: the permutation is a register renaming)
template <int LR>
__device__ __forceinline__ void dft_fwd(float2* v)
{
    constexpr int R = 1 << LR;
    float2 w[R];
#pragma unroll
    for (int j = 0; j < R; j++) w[brev(j, LR)] = v[j];
    if constexpr (LR >= 1) dit_const_stage<R, -1, 1, true>(w);
    if constexpr (LR >= 2) dit_const_stage<R, -1, 2, true>(w);
    if constexpr (LR >= 3) dit_const_stage<R, -1, 3, true>(w);
    if constexpr (LR >= 4) dit_const_stage<R, -1, 4, true>(w);
#pragma unroll
    for (int j = 0; j < R; j++) v[j] = w[j];
}

struct SpecColArgs {
    int n_col_tiles;        // tiles along the contiguous index, per outer index
    int n_outer;            // outer indices per batch entry (1 in pass A, Ra in pass B)
    int xs;                 // twiddle W_D^{x y}: x = column >> xs
    int y0_mul, ymul;       //                     y = y0_mul * outer + ymul * row
    int logD;
    int store_rows_outer;   // 0: store box (T, R, 1) at (c0, 0, o)  [pass A];  1: box (T, 1, R) at (c0, outer, batch R) [pass B]
    double* part;           // pass A: per-tile partial sums [batch][n_tiles][3], else NULL
    uint32_t* status;       // device status word (mbarrier time-outs)
};

// Column pass: tile = R rows x T = 4096/R contiguous columns; thread (c = tid % T, t = tid / T) of P = R/16.
//   stage 1: 16-point DFT over j of rows t + P j, twiddle W_R^{t r}, written back to row t + P r (its own slots);
//   stage 2: rows 16 t + i, i = 0..15 hold Y_{i mod P}[r = (16 t + i)/P]: 16/P DFTs of length P give the outputs
//            k = r + 16 q; times the pass twiddle; to the second tile, which one box store sends out.
template <int LR, bool ACC_POWER>
__global__ void __launch_bounds__(SPT_THREADS, 3)
k_spec_cols(const __grid_constant__ CUtensorMap in, const __grid_constant__ CUtensorMap out, SpecColArgs a)
{
    constexpr int R = 1 << LR, P = R / 16, LP = LR - 4, T = SPT_TILE / R, G = 16 / P;
    extern __shared__ __align__(128) float2 dsm[];
    float2* tin = dsm;                               // [R][T]
    float2* tout = dsm + SPT_TILE;                   // [R][T]
    __shared__ __align__(8) uint64_t bar;
    __shared__ float2 twr[R];                        // W_R^x, x in [0, R)
    __shared__ double red[3][SPT_THREADS];           // pass A only (unused and dropped otherwise)
    const int tid = threadIdx.x, c = tid % T, t = tid / T;
    const int bt = blockIdx.y;
    const int outer = blockIdx.x / a.n_col_tiles, c0 = (blockIdx.x - outer * a.n_col_tiles) * T;
    if (tid == 0) {
        mbar_init(&bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&bar, SPT_TILE_BYTES);
        tma_load_3d(tin, &in, c0, 0, bt * a.n_outer + outer, &bar);
    }
    if (tid < R) twr[tid] = twiddle(tid, R, -1.0f);  // overlaps the copy
    if (!mbar_wait(&bar, 0, a.status)) return;

    float2 v[16];
#pragma unroll
    for (int j = 0; j < 16; j++) v[j] = tin[(t + P * j) * T + c];
    if constexpr (ACC_POWER) {
        double s1 = 0.0, s2 = 0.0, sa = 0.0;
#pragma unroll
        for (int j = 0; j < 16; j++) {
            const double x = v[j].x, y = v[j].y;
            s1 += x + y;
            sa += x - y;
            s2 = fma(x, x, fma(y, y, s2));
        }
        red[0][tid] = s1; red[1][tid] = s2; red[2][tid] = sa;
    }
    dft_fwd<4>(v);
    __syncthreads();                                 // twr complete (and red written)
#pragma unroll
    for (int r = 0; r < 16; r++) {
        const float2 y = (r == 0) ? v[0] : cmul(v[r], twr[t * r]);
        tin[(t + P * r) * T + c] = y;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; i++) v[i] = tin[(16 * t + i) * T + c];
    // pass twiddle W_D^{x y}, y = y0 + ymul k, k = r + 16 q:  W^{x (y0 + ymul r)} (W^{16 x ymul})^q -- one sincospif
    // per group and one for the step, whose powers come from products of depth <= 4 (a few 1e-8 of extra error);
    // every exponent is reduced mod D as an integer first and is exact in fp32 (D <= 2^24)
    const int col = c0 + c;
    const unsigned x = (unsigned)col >> a.xs, y0 = (unsigned)(a.y0_mul * outer), dmask = (1u << a.logD) - 1u;
    const float dinv = 2.0f / (float)(1u << a.logD);
    float2 st[P];                                     // st[q] = step^q
    st[0] = make_float2(1.0f, 0.0f);
    {
        const unsigned e = (16u * x * (unsigned)a.ymul) & dmask;
        float sn, cs;
        sincospif((float)e * dinv, &sn, &cs);
        st[1] = make_float2(cs, -sn);
#pragma unroll
        for (int q = 2; q < P; q++) st[q] = cmul(st[q >> 1], st[q - (q >> 1)]);
    }
#pragma unroll
    for (int g = 0; g < G; g++) {
        dft_fwd<LP>(v + g * P);
        const int r = G * t + g;
        const unsigned e = (x * (y0 + (unsigned)(a.ymul * r))) & dmask;
        float sn, cs;
        sincospif((float)e * dinv, &sn, &cs);
        const float2 base = make_float2(cs, -sn);
#pragma unroll
        for (int q = 0; q < P; q++)
            tout[(r + 16 * q) * T + c] = cmul(v[g * P + q], q == 0 ? base : cmul(base, st[q]));
    }
    fence_proxy_async();
    if constexpr (ACC_POWER) {                        // fixed-order tree over the CTA (deterministic)
        for (int o = SPT_THREADS / 2; o > 0; o >>= 1) {
            __syncthreads();
            if (tid < o)
                for (int q = 0; q < 3; q++) red[q][tid] += red[q][tid + o];
        }
    }
    __syncthreads();                                 // tout and the sums are complete
    if constexpr (ACC_POWER) {
        if (tid < 3) a.part[((size_t)bt * gridDim.x + blockIdx.x) * 3 + tid] = red[tid][0];
    }
    if (tid == 0) {
        if (a.store_rows_outer) tma_store_3d(&out, tout, c0, outer, bt * R);
        else tma_store_3d(&out, tout, c0, 0, bt * a.n_outer + outer);
        tma_store_commit();
        tma_store_wait_all();
    }
}

// mu and 1/sqrt(mu) of every series from the per-tile sums of pass A, same order for every run.
// grid = n_batch, block = 256.  scale[b] = 0 for the all-zero series (G22).
__global__ void __launch_bounds__(256)
k_spec_scale(const double* __restrict__ part, int n_part, int M, float* __restrict__ scale, float* __restrict__ meanpow)
{
    __shared__ double red[3][256];
    const int bt = blockIdx.x;
    double acc[3] = {0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < n_part; i += blockDim.x)
        for (int q = 0; q < 3; q++) acc[q] += part[((size_t)bt * n_part + i) * 3 + q];
    for (int q = 0; q < 3; q++) red[q][threadIdx.x] = acc[q];
    for (int o = 128; o > 0; o >>= 1) {
        __syncthreads();
        if ((int)threadIdx.x < o)
            for (int q = 0; q < 3; q++) red[q][threadIdx.x] += red[q][threadIdx.x + o];
    }
    if (threadIdx.x == 0) {
        const double N = 2.0 * (double)M;
        const double tot = 0.5 * (N * red[1][0] - red[0][0] * red[0][0] + red[2][0] * red[2][0]);
        const double mu = tot / (double)M;
        scale[bt] = mu > 0.0 ? (float)(1.0 / sqrt(mu)) : 0.0f;
        if (meanpow) meanpow[bt] = (float)mu;
    }
}

struct SpecRowArgs {
    const float2* src;      // [batch][NR][Rc]  rows in natural frequency order kappa
    float2* spec;           // [batch][M]       S[c] = F_{c+1} * scale
    const float* scale;     // [batch]
    int NR, M;
    uint32_t* status;
};

// Row pass: item i of a batch entry = rows A_j = i T/2 + j and their partners B_j = NR - A_j (j < T/2); in item 0
// row 0 pairs with itself and its partner slot carries the other self-paired row, NR/2.  T = 4096/Rc rows, thread
// (rho = tid / P, t = tid % P), P = Rc/16.  Rows sit at a pitch of Rc + 2 values (bulk-copy destinations stay
// 16-byte aligned, and the untangle's reads down a column of pairs are conflict-free); the exchange between
// the two DFT stages uses a pitch of 17 per 16 values.
template <int LR>
__global__ void __launch_bounds__(SPT_THREADS, 3)
k_spec_rows(SpecRowArgs a)
{
    constexpr int R = 1 << LR, P = R / 16, LP = LR - 4, T = SPT_TILE / R, G = 16 / P, H = T / 2;
    constexpr int PITCH = R + 2, XP = R + R / 16;
    extern __shared__ __align__(128) float2 dsm[];
    float2* tin = dsm;                               // [T][PITCH]: the rows, later their transforms
    float2* ex = dsm + T * PITCH;                    // [T][XP]
    __shared__ __align__(8) uint64_t bar;
    __shared__ float2 twr[R];                        // W_R^x
    __shared__ float2 twu[R];                        // W_{2R}^x = W_N^{NR x}: the k_c part of the untangle twiddle
    const int tid = threadIdx.x, rho = tid / P, t = tid % P;
    const int bt = blockIdx.y, item = blockIdx.x;
    const int NR = a.NR, M = a.M;
    auto row_of = [&](int slot) {                    // slot < H: A_j; else B_j
        const int j = slot < H ? slot : slot - H, ka = item * H + j;
        return slot < H ? ka : (ka == 0 ? NR / 2 : NR - ka);
    };
    if (tid == 0) {
        mbar_init(&bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&bar, SPT_TILE_BYTES);
        const float2* base = a.src + (size_t)bt * M;
        for (int s = 0; s < T; s++) tma_load_1d(tin + s * PITCH, base + (size_t)row_of(s) * R, R * 8, &bar);
    }
    if (tid < R) {
        twr[tid] = twiddle(tid, R, -1.0f);
        twu[tid] = twiddle(tid, 2 * R, -1.0f);
    }
    if (!mbar_wait(&bar, 0, a.status)) return;

    float2 v[16];
#pragma unroll
    for (int j = 0; j < 16; j++) v[j] = tin[rho * PITCH + t + P * j];
    dft_fwd<4>(v);
    __syncthreads();                                 // twr complete; every row has been read
#pragma unroll
    for (int r = 0; r < 16; r++) {
        const int s = t + P * r;
        ex[rho * XP + s + (s >> 4)] = (r == 0) ? v[0] : cmul(v[r], twr[t * r]);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; i++) v[i] = ex[rho * XP + 17 * t + i];
#pragma unroll
    for (int g = 0; g < G; g++) {
        dft_fwd<LP>(v + g * P);
#pragma unroll
        for (int q = 0; q < P; q++) tin[rho * PITCH + (G * t + g) + 16 * q] = v[g * P + q];
    }
    __syncthreads();

    // untangle: thread (pair = tid % H, kk = tid / H) walks k_c = kk, kk + 256/H, ...
    const float sc = a.scale[bt];
    float2* out = a.spec + (size_t)bt * M;
    const int pr = tid % H, ka = item * H + pr;
    const float2* ra = tin + pr * PITCH;             // row kappa
    const float2* rb = tin + (H + pr) * PITCH;       // its partner (or, for kappa = 0, row NR/2)
    // W_N^k, k = kappa + NR kc, as W_N^kappa (one sincospif per thread) times W_{2 Rc}^kc (table): N = 2 NR Rc
    const int N = 2 * M;
    const float2 wka = twiddle(ka, N, -1.0f), whalf = twiddle(1, 4 * R, -1.0f);     // W_N^{NR/2} = W_{4 Rc}
    for (int kc = tid / H; kc < R; kc += SPT_THREADS / H) {
        if (ka != 0) {
            const float2 za = ra[kc], zb = rb[R - 1 - kc];           // Z_k, Z_{M-k},  k = kappa + NR kc
            const int k = ka + NR * kc;
            const float2 e = make_float2(0.5f * (za.x + zb.x), 0.5f * (za.y - zb.y));       // (Z_k + conj Z_{M-k})/2
            const float2 d = make_float2(0.5f * (za.x - zb.x), 0.5f * (za.y + zb.y));       // (Z_k - conj Z_{M-k})/2
            const float2 p = cmul(make_float2(d.y, -d.x), cmul(wka, twu[kc]));               // W_N^k O_k,  O = -i d
            out[k - 1] = make_float2((e.x + p.x) * sc, (e.y + p.y) * sc);                  // F_k
            out[M - k - 1] = make_float2((e.x - p.x) * sc, -(e.y - p.y) * sc);             // F_{M-k} = conj(E - W O)
        } else {
            // row 0 (k = NR kc, partner (Rc - kc) mod Rc in the same row) and row NR/2 (k = NR/2 + NR kc, partner Rc-1-kc)
            const float2 z0 = ra[kc], z0p = ra[(R - kc) & (R - 1)];
            if (kc == 0) {
                out[M - 1] = make_float2((z0.x - z0.y) * sc, 0.0f);                        // Nyquist; DC is dropped
            } else {
                const int k = NR * kc;
                const float2 e = make_float2(0.5f * (z0.x + z0p.x), 0.5f * (z0.y - z0p.y));
                const float2 d = make_float2(0.5f * (z0.x - z0p.x), 0.5f * (z0.y + z0p.y));
                const float2 p = cmul(make_float2(d.y, -d.x), twu[kc]);                       // k = NR kc
                out[k - 1] = make_float2((e.x + p.x) * sc, (e.y + p.y) * sc);
            }
            const float2 zh = rb[kc], zhp = rb[R - 1 - kc];
            const int k = NR / 2 + NR * kc;
            const float2 e = make_float2(0.5f * (zh.x + zhp.x), 0.5f * (zh.y - zhp.y));
            const float2 d = make_float2(0.5f * (zh.x - zhp.x), 0.5f * (zh.y + zhp.y));
            const float2 p = cmul(make_float2(d.y, -d.x), cmul(whalf, twu[kc]));              // k = NR/2 + NR kc
            out[k - 1] = make_float2((e.x + p.x) * sc, (e.y + p.y) * sc);
        }
    }
}

// ------------------------------------------------------------------ host
bool fdas_spectrum_tma_supported(const fdas_plan* p) { return p->sp_npass != 0; }

// M = 2^m into two or three factors of 2^5 .. 2^8 (m >= 12), the contiguous one (Rc) as long as possible.
void fdas_spectrum_tma_plan(fdas_plan* p)
{
    int m = 0;
    while ((1LL << m) < p->M) m++;
    p->sp_npass = 0;
    if (m < 12) return;
    if (m <= 16) {
        p->sp_npass = 2;
        p->sp_lc = (m + 1) / 2 < 8 ? (m + 1) / 2 : 8;
        p->sp_la = m - p->sp_lc;
        p->sp_lb = 0;
    } else {
        p->sp_npass = 3;
        p->sp_lc = m >= 18 ? 8 : 7;
        const int rest = m - p->sp_lc;
        p->sp_la = (rest + 1) / 2;
        p->sp_lb = rest / 2;
    }
}

template <int LR, bool ACC>
static int launch_cols(const CUtensorMap& in, const CUtensorMap& out, const SpecColArgs& a, int n_batch, cudaStream_t st)
{
    const int smem = 2 * SPT_TILE_BYTES;
    FDAS_CUDA(cudaFuncSetAttribute(k_spec_cols<LR, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    FDAS_CUDA(cudaFuncSetAttribute(k_spec_cols<LR, ACC>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));   // 3 CTAs x 72 KB
    k_spec_cols<LR, ACC><<<dim3(a.n_outer * a.n_col_tiles, n_batch), SPT_THREADS, smem, st>>>(in, out, a);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}
template <bool ACC>
static int launch_cols_lr(int lr, const CUtensorMap& in, const CUtensorMap& out, const SpecColArgs& a, int n_batch, cudaStream_t st)
{
    switch (lr) {
    case 5: return launch_cols<5, ACC>(in, out, a, n_batch, st);
    case 6: return launch_cols<6, ACC>(in, out, a, n_batch, st);
    case 7: return launch_cols<7, ACC>(in, out, a, n_batch, st);
    case 8: return launch_cols<8, ACC>(in, out, a, n_batch, st);
    default: return FDAS_E_INVALID;
    }
}
template <int LR>
static int launch_rows(const SpecRowArgs& a, int n_batch, cudaStream_t st)
{
    constexpr int R = 1 << LR, T = SPT_TILE / R;
    const int smem = (T * (R + 2) + T * (R + R / 16)) * 8;          // a multiple of 128 for every R here
    FDAS_CUDA(cudaFuncSetAttribute(k_spec_rows<LR>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    FDAS_CUDA(cudaFuncSetAttribute(k_spec_rows<LR>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    k_spec_rows<LR><<<dim3(a.NR / T, n_batch), SPT_THREADS, smem, st>>>(a);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}

// d_ws: [ws_inter_bytes: M complex per batch entry][ws_part_bytes: partial sums, then one scale per batch entry]
int fdas_launch_spectrum_tma(fdas_plan* p, const float* d_series, int n_batch, float2* d_spec, float* d_meanpow, void* d_ws,
                             cudaStream_t st)
{
    const int la = p->sp_la, lb = p->sp_lb, lc = p->sp_lc;
    const uint64_t Ra = 1ull << la, Rb = 1ull << lb, Rc = 1ull << lc, M = (uint64_t)p->M;
    float2* inter = reinterpret_cast<float2*>(d_ws);
    double* part = reinterpret_cast<double*>(reinterpret_cast<char*>(d_ws) + p->ws_inter_bytes);
    const int n_part = (int)(M / SPT_TILE);
    float* scale = reinterpret_cast<float*>(part + (size_t)p->max_batch * n_part * 3);
    uint32_t* status = p->d_status;
    const uint64_t nb = (uint64_t)n_batch;
    CUtensorMap mi, mo;
    SpecColArgs ca;
    // ---- pass A: [batch][Ra][Rb Rc] -> same shape; three passes: into the spectrum buffer, two passes: into the workspace
    float2* dstA = p->sp_npass == 3 ? d_spec : inter;
    {
        const uint64_t C = Rb * Rc;
        const uint64_t dims[3] = {C, Ra, nb}, str[2] = {C * 8, M * 8};
        const uint32_t box[3] = {(uint32_t)(SPT_TILE >> la), (uint32_t)Ra, 1};
        if (!fdas_encode_tensor_map(&mi, d_series, 3, dims, str, box) || !fdas_encode_tensor_map(&mo, dstA, 3, dims, str, box))
            return FDAS_E_INVALID;
        ca.n_col_tiles = (int)(C >> (12 - la)); ca.n_outer = 1;
        ca.xs = p->sp_npass == 3 ? lc : 0; ca.y0_mul = 0; ca.ymul = 1; ca.logD = p->sp_npass == 3 ? la + lb : la + lc;
        ca.store_rows_outer = 0; ca.part = part; ca.status = status;
        int rc = launch_cols_lr<true>(la, mi, mo, ca, n_batch, st);
        if (rc) return rc;
    }
    k_spec_scale<<<n_batch, 256, 0, st>>>(part, n_part, (int)M, scale, d_meanpow);
    FDAS_LAUNCH_CHECK();
    // ---- pass B: for every k_a, [Rb][Rc] -> rows kappa = k_a + Ra k_b of [Ra Rb][Rc] in the workspace
    if (p->sp_npass == 3) {
        const uint64_t di[3] = {Rc, Rb, Ra * nb}, si[2] = {Rc * 8, Rb * Rc * 8};
        const uint32_t bi[3] = {(uint32_t)(SPT_TILE >> lb), (uint32_t)Rb, 1};
        const uint64_t dO[3] = {Rc, Ra, Rb * nb}, so[2] = {Rc * 8, Ra * Rc * 8};
        const uint32_t bo[3] = {(uint32_t)(SPT_TILE >> lb), 1, (uint32_t)Rb};
        if (!fdas_encode_tensor_map(&mi, d_spec, 3, di, si, bi) || !fdas_encode_tensor_map(&mo, inter, 3, dO, so, bo))
            return FDAS_E_INVALID;
        ca.n_col_tiles = (int)(Rc >> (12 - lb)); ca.n_outer = (int)Ra;
        ca.xs = 0; ca.y0_mul = 1; ca.ymul = (int)Ra; ca.logD = la + lb + lc;
        ca.store_rows_outer = 1; ca.part = nullptr; ca.status = status;
        int rc = launch_cols_lr<false>(lb, mi, mo, ca, n_batch, st);
        if (rc) return rc;
    }
    // ---- pass C
    SpecRowArgs ra;
    ra.src = inter; ra.spec = d_spec; ra.scale = scale; ra.NR = (int)(Ra * Rb); ra.M = (int)M; ra.status = status;
    switch (lc) {
    case 6: return launch_rows<6>(ra, n_batch, st);
    case 7: return launch_rows<7>(ra, n_batch, st);
    case 8: return launch_rows<8>(ra, n_batch, st);
    default: return FDAS_E_INVALID;
    }
}

// ------------------------------------------------------------------ init-stage self-test
// The TMA-staged passes have a second, independent implementation of the same transform next to them (the generic
// kernels).  At plan build -- the "initialization stage", outside every timed region -- both transform
// one seeded pseudo-random series of the plan's own length and the results are compared on the device.  If the
// asynchronous-copy path disagrees or one of its waits timed out (a wrong tensor map, a byte count: mistakes that
// no CPU run can exclude), the plan says so in its status word (FDAS_STATUS_TMA_FALLBACK) and uses the generic
// kernels from then on: a defect costs speed and is reported, it does not silently corrupt a search.
__global__ void __launch_bounds__(256)
k_selftest_fill(float* __restrict__ x, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        unsigned h = (unsigned)i * 2654435761u;
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
        float s, c;
        sincospif(2.0f * (float)(i & 1023) * (37.0f / 1024.0f), &s, &c);
        x[i] = (float)(h >> 8) * (1.0f / 8388608.0f) - 1.0f + 0.25f * c;
    }
}
__global__ void __launch_bounds__(256)
k_selftest_diff(const float* __restrict__ a, const float* __restrict__ b, long long n, unsigned* __restrict__ worst)
{
    float m = 0.0f;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float d = fabsf(a[i] - b[i]);
        m = (d == d) ? fmaxf(m, d) : 3.0e38f;                          // a NaN counts as the worst possible
    }
    atomicMax(worst, __float_as_uint(m));                               // non-negative floats order like their bit patterns
}

// mode: 0 = run, 2 = pretend the comparison failed (test hook).  Out of memory: the test is skipped.
int fdas_spectrum_selftest(fdas_plan* p, int mode, cudaStream_t st)
{
    if (!p->sp_npass || !p->d_status) return FDAS_OK;
    const size_t N = (size_t)p->n_samples, M = (size_t)p->M;
    float* x = nullptr; float2* s1 = nullptr; float2* s2 = nullptr; void* ws = nullptr; unsigned* worst = nullptr;
    bool mem = cudaMalloc(&x, N * 4) == cudaSuccess && cudaMalloc(&s1, M * 8) == cudaSuccess && cudaMalloc(&s2, M * 8) == cudaSuccess &&
               cudaMalloc(&ws, p->workspace_bytes) == cudaSuccess && cudaMalloc(&worst, 4) == cudaSuccess;
    int rc = FDAS_OK;
    unsigned h_worst = 0, h_status = 0;
    if (mem) {
        cudaMemsetAsync(worst, 0, 4, st);
        k_selftest_fill<<<592, 256, 0, st>>>(x, (long long)N);
        rc = fdas_launch_spectrum_tma(p, x, 1, s1, nullptr, ws, st);
        if (rc == FDAS_OK) rc = fdas_launch_spectrum(p, x, 1, s2, nullptr, ws, st);
        if (rc == FDAS_OK) {
            k_selftest_diff<<<592, 256, 0, st>>>(reinterpret_cast<const float*>(s1), reinterpret_cast<const float*>(s2), (long long)(2 * M), worst);
            if (cudaMemcpyAsync(&h_worst, worst, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaMemcpyAsync(&h_status, p->d_status, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess)
                rc = FDAS_E_CUDA;
        }
    } else {
        cudaGetLastError();
    }
    if (x) cudaFree(x);
    if (s1) cudaFree(s1);
    if (s2) cudaFree(s2);
    if (ws) cudaFree(ws);
    if (worst) cudaFree(worst);
    if (rc == FDAS_E_CUDA) { fdas_set_cuda_error(cudaGetLastError(), "fdas_spectrum_selftest"); return rc; }
    if (!mem || rc != FDAS_OK) return FDAS_OK;                          // could not be run: nothing is concluded
    float worst_f;
    memcpy(&worst_f, &h_worst, 4);
    // both paths are within ~1e-6 of the exact spectrum (|S| ~ 1 after normalisation): 1e-3 is far outside rounding
    const bool bad = mode == 2 || (h_status & FDAS_STATUS_MBAR_TIMEOUT) || !(worst_f < 1.0e-3f);
    const uint32_t word = bad ? FDAS_STATUS_TMA_FALLBACK : 0u;
    if (bad) p->tune_spec_generic = 1;
    FDAS_CUDA(cudaMemcpyAsync(p->d_status, &word, 4, cudaMemcpyHostToDevice, st));
    FDAS_CUDA(cudaStreamSynchronize(st));
    return FDAS_OK;
}

int fdas_occupancy_spectrum(int which, int32_t* ctas, int32_t* regs, int32_t* smem)
{
    if (which == 0) return fdas_occupancy_of(k_spec_cols<7, true>, SPT_THREADS, 2 * SPT_TILE_BYTES, ctas, regs, smem);
    if (which == 1) return fdas_occupancy_of(k_spec_cols<7, false>, SPT_THREADS, 2 * SPT_TILE_BYTES, ctas, regs, smem);
    return fdas_occupancy_of(k_spec_rows<8>, SPT_THREADS, (16 * 258 + 16 * 272) * 8, ctas, regs, smem);
}
