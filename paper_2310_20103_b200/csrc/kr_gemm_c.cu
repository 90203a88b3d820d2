// Complex FP64 tensor-core GEMMs of the periodic Tamm-Dancoff operator
//   A(q) x = Delta o x + K^H ( V ( K x ) ),   K[mu, (k, v, c)] = conj(psi_{v k}(mu)) psi_{c k+q}(mu)
// with K never formed:
//   MODE_FWD  T[b][mu]        = sum_{k v} conj(psi_vk[mu]) sum_c psi_ck+q[mu][c] x[b][k][v][c]
//   MODE_BWD  U[b][k][v][c]   = sum_mu psi_vk[mu] conj(psi_ck+q[mu][c]) W[b][mu]
// (the V product in between is the REAL plain GEMM of kr_gemm.cu on the two planes of T: V is real symmetric).
//
// Every array is PLANAR (a real plane and an imaginary plane), so that the complex multiply-add becomes four real
// DMMAs on fragments that sit at the same shared-memory position of the two planes:
//   a = s (*) A   (s = conj(psi_v) on rows in FWD, psi_v on k in BWD with A conjugated): a_r = s_r A_r + s_i A_i,
//   t = s_r A_i - s_i A_r (= +Im a in FWD, -Im a in BWD), formed in registers (2 + 2 FP64 ops per A fragment pair);
//   FWD: out_r += a_r b_r + t (-b_i), out_i += a_r b_i + t b_r;   BWD: out_r += a_r b_r + t b_i, out_i += a_r b_i + t (-b_r).
// 4 real multiply-adds per complex one, the minimum; 64 DMMAs per k-step of a 32x32 warp tile against 16 LDS.64.
// Same pipeline as kr_gemm.cu: one producer warpgroup (one elected lane issues the TMA loads of a stage: two A planes,
// two B planes, two scale planes), 8 consumer warps, "full"/"empty" mbarriers per stage, no CTA-wide barrier in the loop.
#include <algorithm>

#include "kr_gemm_common.cuh"

namespace gwl {

namespace {

template <int BM, int BN, int MODE>
struct TileCfgC {
    static constexpr int A_BYTES = BM * 128;  // per plane
    static constexpr int B_BYTES = BN * 128;
    static constexpr int SC_BYTES = MODE == MODE_FWD ? BM * 8 : 128;
    static constexpr int TX_BYTES = 2 * (A_BYTES + B_BYTES + SC_BYTES);
    static constexpr int KT_BYTES = (TX_BYTES + 1023) / 1024 * 1024;
};

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
        : "memory");
}

template <int BM, int BN, int STAGES, int MODE, int EPI>
__global__ void __launch_bounds__(((BM / 32) * (BN / 32) + 4) * 32, 1)
    gemm_tn_zmma(const GemmParamsC p, const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                 const __grid_constant__ CUtensorMap tmS) {
    constexpr int WM = 32, WN = 32;
    constexpr int WGM = BM / WM, WGN = BN / WN;
    constexpr int NCW = WGM * WGN;
    constexpr int FM = WM / 8, FN = WN / 8;
    constexpr bool FWD = MODE == MODE_FWD;
    using TC = TileCfgC<BM, BN, MODE>;

    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[2 * STAGES];
    __shared__ double red[(EPI == EPI_STORE) ? 1 : WGM * BN];
    const uint32_t smem_base = (static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)) + 1023u) & ~1023u;
    unsigned char* smem_gen = smem_raw + (smem_base - static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)));
    const uint32_t bar_base = static_cast<uint32_t>(__cvta_generic_to_shared(bars));
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp % WGM, wn = (warp / WGM) % WGN;
    const int g = lane >> 2, q = lane & 3;
    const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN, z = blockIdx.z;
    // FWD: z = split over the (k, v, c-tile) reduction; BWD: z = kv (pair of k-point and occupied orbital)
    const int KT = p.kt_total;
    const int kb = FWD ? min(z * p.kt_per_split, KT) : 0;
    const int ke = FWD ? min(kb + p.kt_per_split, KT) : KT;
    const int kpt = FWD ? 0 : z / p.n_v;  // BWD: k-point of this kv

    if (tid == 0) {
        tma_prefetch_desc(&tmA);
        tma_prefetch_desc(&tmB);
        tma_prefetch_desc(&tmS);
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), NCW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    pdl_trigger();
    pdl_wait();

    if (warp >= NCW) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
        if (warp == NCW && lane == 0) {
            int it = 0;
            for (int kt = kb; kt < ke; ++kt, ++it) {
                const int slot = it % STAGES;
                const uint32_t par = ((it / STAGES) & 1) ^ 1;
                while (!mbar_try_wait(empty_bar(slot), par)) {
                }
                const uint32_t fb = full_bar(slot);
                mbar_expect_tx(fb, TC::TX_BYTES);
                const uint32_t sAr = smem_base + slot * TC::KT_BYTES;
                const uint32_t sAi = sAr + TC::A_BYTES;
                const uint32_t sBr = sAi + TC::A_BYTES;
                const uint32_t sBi = sBr + TC::B_BYTES;
                const uint32_t sSr = sBi + TC::B_BYTES;
                const uint32_t sSi = sSr + TC::SC_BYTES;
                if (FWD) {
                    // k-tile order (k-point, c-tile, v): the A tile is the same for n_v consecutive k-tiles (L2 hit)
                    const int per_k = p.a_wrap * p.n_v;
                    const int kp = kt / per_k, rem = kt - kp * per_k;
                    const int ct = rem / p.n_v, kv = kp * p.n_v + (rem - ct * p.n_v);
                    const int a_col = (kp * p.a_wrap + ct) * BK;  // the conduction block of this k-point
                    const int b_col = (kv * p.a_wrap + ct) * BK;
                    tma_load_3d(sAr, &tmA, a_col, m0, 0, fb);
                    tma_load_3d(sAi, &tmA, a_col, m0, 1, fb);
                    tma_load_2d(sBr, &tmB, b_col, n0, fb);                     // x planes: column offset n_kv * n_cp apart
                    tma_load_2d(sBi, &tmB, p.b_plane_cols + b_col, n0, fb);
                    tma_load_3d(sSr, &tmS, m0, kv, 0, fb);
                    tma_load_3d(sSi, &tmS, m0, kv, 1, fb);
                } else {
                    tma_load_3d(sAr, &tmA, kt * BK, kpt * p.n_c + m0, 0, fb);
                    tma_load_3d(sAi, &tmA, kt * BK, kpt * p.n_c + m0, 1, fb);
                    tma_load_3d(sBr, &tmB, kt * BK, n0, 0, fb);
                    tma_load_3d(sBi, &tmB, kt * BK, n0, 1, fb);
                    tma_load_3d(sSr, &tmS, kt * BK, z, 0, fb);
                    tma_load_3d(sSi, &tmS, kt * BK, z, 1, fb);
                }
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;\n");

    double accr[FM][FN][2], acci[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) accr[i][j][0] = accr[i][j][1] = acci[i][j][0] = acci[i][j][1] = 0.0;

    const int xr0 = (2 * (g & 3)), xr1 = xr0 | 1;
    int rowA[FM], rowB[FN];
#pragma unroll
    for (int i = 0; i < FM; ++i) rowA[i] = wm * WM + 16 * (i >> 1) + 2 * g + (i & 1);
#pragma unroll
    for (int j = 0; j < FN; ++j) rowB[j] = wn * WN + 16 * (j >> 1) + 2 * g + (j & 1);

    int it = 0;
    for (int kt = kb; kt < ke; ++kt, ++it) {
        const int slot = it % STAGES;
        const uint32_t par = (it / STAGES) & 1;
        while (!mbar_try_wait(full_bar(slot), par)) {
        }
        const unsigned char* base = smem_gen + slot * TC::KT_BYTES;
        const double* Ar = reinterpret_cast<const double*>(base);
        const double* Ai = reinterpret_cast<const double*>(base + TC::A_BYTES);
        const double* Br = reinterpret_cast<const double*>(base + 2 * TC::A_BYTES);
        const double* Bi = reinterpret_cast<const double*>(base + 2 * TC::A_BYTES + TC::B_BYTES);
        const double* Sr = reinterpret_cast<const double*>(base + 2 * TC::A_BYTES + 2 * TC::B_BYTES);
        const double* Si = reinterpret_cast<const double*>(base + 2 * TC::A_BYTES + 2 * TC::B_BYTES + TC::SC_BYTES);
        double sr[FM], si[FM];
        if (FWD) {
#pragma unroll
            for (int i = 0; i < FM; ++i) {
                sr[i] = Sr[rowA[i]];
                si[i] = Si[rowA[i]];
            }
        }
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
            const int ch = 2 * ks + (q >> 1);
            const int c0 = ((ch ^ xr0) << 1) | (q & 1);
            const int c1 = ((ch ^ xr1) << 1) | (q & 1);
            double a[FM], t[FM], br[FN], bi[FN], nb[FN];
            double skr = 0.0, ski = 0.0;
            if (!FWD) {
                skr = Sr[4 * ks + q];
                ski = Si[4 * ks + q];
            }
#pragma unroll
            for (int i = 0; i < FM; ++i) {
                const int off = rowA[i] * 16 + ((i & 1) ? c1 : c0);
                const double xr_ = Ar[off], xi_ = Ai[off];
                const double s_r = FWD ? sr[i] : skr, s_i = FWD ? si[i] : ski;
                a[i] = fma(s_r, xr_, s_i * xi_);
                t[i] = fma(s_r, xi_, -(s_i * xr_));
            }
#pragma unroll
            for (int j = 0; j < FN; ++j) {
                const int off = rowB[j] * 16 + ((j & 1) ? c1 : c0);
                br[j] = Br[off];
                bi[j] = Bi[off];
                nb[j] = FWD ? -bi[j] : -br[j];
            }
            // two passes so that the two DMMAs into one accumulator are 32 instructions apart
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) {
                    dmma_8x8x4(accr[i][j][0], accr[i][j][1], a[i], br[j]);
                    dmma_8x8x4(acci[i][j][0], acci[i][j][1], a[i], bi[j]);
                }
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) {
                    dmma_8x8x4(accr[i][j][0], accr[i][j][1], t[i], FWD ? nb[j] : bi[j]);
                    dmma_8x8x4(acci[i][j][0], acci[i][j][1], t[i], FWD ? br[j] : nb[j]);
                }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar(slot));
    }

    // ---- epilogue: acc[i][j][e] is row m0 + rowA[i] (i even/odd adjacent), column n0 + wn*WN + 16*(j>>1) + 2*(2q+e) + (j&1)
    if (EPI == EPI_STORE) {
        double* outr = p.out + (int64_t)z * p.out_split_stride;
        double* outi = outr + p.o_plane;
        const bool vec_ok = ((p.ldo & 1) == 0) && ((p.o_plane & 1) == 0) && ((p.out_split_stride & 1) == 0) &&
                            ((reinterpret_cast<uintptr_t>(p.out) & 15) == 0);
#pragma unroll
        for (int i2 = 0; i2 < FM / 2; ++i2) {
            const int r0 = m0 + wm * WM + 16 * i2 + 2 * g;
#pragma unroll
            for (int j = 0; j < FN; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                    if (n >= p.N) continue;
                    const int64_t off = (int64_t)n * p.ldo + r0;
                    if (vec_ok && r0 + 1 < p.M) {
                        *reinterpret_cast<double2*>(outr + off) = make_double2(accr[2 * i2][j][e], accr[2 * i2 + 1][j][e]);
                        *reinterpret_cast<double2*>(outi + off) = make_double2(acci[2 * i2][j][e], acci[2 * i2 + 1][j][e]);
                    } else {
                        if (r0 < p.M) {
                            outr[off] = accr[2 * i2][j][e];
                            outi[off] = acci[2 * i2][j][e];
                        }
                        if (r0 + 1 < p.M) {
                            outr[off + 1] = accr[2 * i2 + 1][j][e];
                            outi[off + 1] = acci[2 * i2 + 1][j][e];
                        }
                    }
                }
        }
        return;
    }
    // BWD: y = d2 o x + coupling u (EPI_CASIDA; TDA: d2 = Delta, coupling 1) or y = u (EPI_START), both planes, and the
    // per-column partial sums of Re<x, y> (alpha) or <y, y> (norm of the start vector)
    const int64_t voff = (int64_t)z * p.n_c;
    const double cpl = p.coupling;
    double part[FN][2];
#pragma unroll
    for (int j = 0; j < FN; ++j) part[j][0] = part[j][1] = 0.0;
#pragma unroll
    for (int i2 = 0; i2 < FM / 2; ++i2) {
        const int r0 = m0 + wm * WM + 16 * i2 + 2 * g;
        if (r0 >= p.M) continue;
        const bool two = (r0 + 1 < p.M);
        double d0 = 0.0, d1 = 0.0;
        if (EPI == EPI_CASIDA) {
            d0 = p.d2[voff + r0];
            d1 = two ? p.d2[voff + r0 + 1] : 0.0;
        }
#pragma unroll
        for (int j = 0; j < FN; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                if (n >= p.N) continue;
                const int64_t off = (int64_t)n * p.ldo + voff + r0;
                double yr0 = cpl * accr[2 * i2][j][e], yr1 = cpl * accr[2 * i2 + 1][j][e];
                double yi0 = cpl * acci[2 * i2][j][e], yi1 = cpl * acci[2 * i2 + 1][j][e];
                if (EPI == EPI_CASIDA) {
                    const int64_t xoff = (int64_t)n * p.ldx + voff + r0;
                    const double xr0v = p.X[xoff], xi0v = p.X[xoff + p.x_plane];
                    const double xr1v = two ? p.X[xoff + 1] : 0.0, xi1v = two ? p.X[xoff + p.x_plane + 1] : 0.0;
                    yr0 = fma(d0, xr0v, yr0);
                    yi0 = fma(d0, xi0v, yi0);
                    yr1 = fma(d1, xr1v, yr1);
                    yi1 = fma(d1, xi1v, yi1);
                    part[j][e] += xr0v * yr0 + xi0v * yi0 + xr1v * yr1 + xi1v * yi1;
                } else {
                    part[j][e] += yr0 * yr0 + yi0 * yi0 + (two ? yr1 * yr1 + yi1 * yi1 : 0.0);
                }
                p.out[off] = yr0;
                p.out[off + p.o_plane] = yi0;
                if (two) {
                    p.out[off + 1] = yr1;
                    p.out[off + p.o_plane + 1] = yi1;
                }
            }
    }
    if (p.dotpart != nullptr) {
        asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");
#pragma unroll
        for (int j = 0; j < FN; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                double vsum = part[j][e];
                vsum += __shfl_xor_sync(0xffffffffu, vsum, 4);
                vsum += __shfl_xor_sync(0xffffffffu, vsum, 8);
                vsum += __shfl_xor_sync(0xffffffffu, vsum, 16);
                if (g == 0) red[wm * BN + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1)] = vsum;
            }
        asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");
        if (tid < BN && n0 + tid < p.N) {
            double ssum = 0.0;
#pragma unroll
            for (int w = 0; w < WGM; ++w) ssum += red[w * BN + tid];
            p.dotpart[(int64_t)(n0 + tid) * p.dot_stride + (int64_t)z * gridDim.x + blockIdx.x] = ssum;
        }
    }
}

// 3-D FP64 tensor map over planar data: [planes][rows][ld] of which `cols` columns are valid
inline cudaError_t make_map3(CUtensorMap* m, const double* base, uint64_t cols, uint64_t rows, uint64_t ld,
                             uint64_t plane_stride, uint32_t box_cols, uint32_t box_rows, bool swizzle) {
    EncodeFn enc = get_encode_fn();
    if (enc == nullptr) return cudaErrorNotSupported;
    cuuint64_t dims[3] = {cols, rows, 2};
    cuuint64_t strides[2] = {ld * sizeof(double), plane_stride * sizeof(double)};
    cuuint32_t box[3] = {box_cols, box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int MODE, int EPI>
cudaError_t launch_c(const GemmParamsC& p, int nz, cudaStream_t st) {
    constexpr int BM = 128, BN = 64, STAGES = 4;
    using TC = TileCfgC<BM, BN, MODE>;
    constexpr int SMEM = STAGES * TC::KT_BYTES + 1024;
    constexpr int NTHREADS = ((BM / 32) * (BN / 32) + 4) * 32;
    static_assert(SMEM <= 227 * 1024, "stage ring does not fit in shared memory");
    auto kern = gemm_tn_zmma<BM, BN, STAGES, MODE, EPI>;
    static SmemAttr attr;
    cudaError_t e = attr.ensure(kern, SMEM);
    if (e != cudaSuccess) return e;
    CUtensorMap tmA, tmB, tmS;
    const uint64_t kcols = (uint64_t)p.kt_total * BK;
    if (MODE == MODE_FWD) {
        // A = psi_cq planar [2][n_mu][n_k * n_cp]; B = xs [nb][2 * n_kv * n_cp] (planes side by side); S = psi_v^T planar
        e = make_map3(&tmA, p.A, (uint64_t)p.lda, (uint64_t)p.M, (uint64_t)p.lda, (uint64_t)p.a_plane, BK, BM, true);
        if (e != cudaSuccess) return e;
        e = make_map(&tmB, p.B, 2 * kcols, (uint64_t)p.N, (uint64_t)p.ldb, BK, BN, true);
        if (e != cudaSuccess) return e;
        e = make_map3(&tmS, p.scale, (uint64_t)p.lds, (uint64_t)p.scale_rows, (uint64_t)p.lds, (uint64_t)p.s_plane, BM, 1, false);
    } else {
        // A = psi_cq^T planar [2][n_k * n_c][n_mup]; B = W planar [2][nb][n_mup]; S = psi_v^T planar
        e = make_map3(&tmA, p.A, kcols, (uint64_t)p.a_rows, (uint64_t)p.lda, (uint64_t)p.a_plane, BK, BM, true);
        if (e != cudaSuccess) return e;
        e = make_map3(&tmB, p.B, kcols, (uint64_t)p.N, (uint64_t)p.ldb, (uint64_t)p.b_plane, BK, BN, true);
        if (e != cudaSuccess) return e;
        e = make_map3(&tmS, p.scale, (uint64_t)p.lds, (uint64_t)p.scale_rows, (uint64_t)p.lds, (uint64_t)p.s_plane, BK, 1, false);
    }
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)ceil_div(p.M, BM), (unsigned)ceil_div(p.N, BN), (unsigned)nz);
    cudaError_t le = launch_pdl(kern, grid, dim3(NTHREADS), SMEM, st, 1u, p, tmA, tmB, tmS);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

}  // namespace

int gemm_c_tiles_m(int M) { return (int)ceil_div(M, 128); }

// Split-K of the FWD product over (k, v, c-tile): same cost model as plan_gemm (waves x (k-tiles per split + fill))
GemmPlan plan_gemm_c(int M, int N, int kt_total, int n_sm) {
    GemmPlan pl;
    pl.bm = 128;
    pl.bn = 64;
    const int64_t tiles = ceil_div(M, pl.bm) * ceil_div(N, pl.bn);
    int64_t best_cost = -1;
    int best_s = 1;
    const int max_s = (int)std::max<int64_t>(1, std::min<int64_t>(64, kt_total / 8));
    for (int s = 1; s <= max_s; ++s) {
        const int64_t kps = ceil_div(kt_total, s);
        const int64_t real_s = ceil_div(kt_total, kps);
        const int64_t waves = ceil_div(tiles * real_s, n_sm);
        const int64_t cost = waves * (kps + 6);
        if (best_cost < 0 || cost < best_cost) {
            best_cost = cost;
            best_s = (int)real_s;
        }
    }
    pl.kt_per_split = (int)ceil_div(kt_total, best_s);
    pl.splits = (int)ceil_div(kt_total, pl.kt_per_split);
    return pl;
}

cudaError_t launch_gemm_c(int mode, int epi, const GemmParamsC& p, int nz, cudaStream_t st) {
    if (p.M <= 0 || p.N <= 0 || nz <= 0) return cudaSuccess;
    if (nz > 65535) return cudaErrorInvalidValue;
    if (mode == MODE_FWD && epi == EPI_STORE) return launch_c<MODE_FWD, EPI_STORE>(p, nz, st);
    if (mode == MODE_BWD && epi == EPI_CASIDA) return launch_c<MODE_BWD, EPI_CASIDA>(p, nz, st);
    if (mode == MODE_BWD && epi == EPI_START) return launch_c<MODE_BWD, EPI_START>(p, nz, st);
    return cudaErrorInvalidValue;
}

}  // namespace gwl
