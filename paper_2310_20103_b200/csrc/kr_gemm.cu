// FP64 tensor-core (DMMA) GEMM core for the three contractions of the Casida product
//   Y = Delta^2 o X + 2 sqrt(Delta) o K^T ( V ( K ( sqrt(Delta) o X ) ) )
// with K[mu, vc] = phi_v(mu) phi_c(mu) never formed (Khatri-Rao structure):
//   MODE_FWD   T[b][mu]   = sum_v phi_v[mu] * sum_c Phi_c[mu][c] Xs[b][v][c]     (row scale applied to the A fragments)
//   MODE_PLAIN W[b][mu]   = sum_nu V[mu][nu] T[b][nu]
//   MODE_BWD   U[b][v][c] = sum_mu Phi_c^T[c][mu] * phi_v[mu] * W[b][mu]          (k scale applied in registers)
// Every product is out[n][m] = sum_k A[m][k] B[n][k], both operands K-contiguous.
//
// sm_100a has no tcgen05 kind for FP64; the FP64 tensor path is the warp-level mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4).
// Tiles are staged in shared memory as 128-byte rows (16 doubles) with the TMA SWIZZLE_128B pattern
// (16-byte chunk index XOR (row & 7)); fragment rows are interleaved (row = 2*g + parity) so that every
// LDS.64 of a half-warp touches 16 distinct 8-byte bank pairs.
#include "gwl_internal.h"

namespace gwl {

thread_local int64_t* g_launch_counter = nullptr;

namespace {

__device__ __forceinline__ void dmma_8x8x4(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
    int sz = valid ? 16 : 0;  // src-size 0 => the 16 destination bytes are zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

template <int BM, int BN, int MODE>
struct TileCfg {
    static constexpr int A_BYTES = BM * 128;
    static constexpr int B_BYTES = BN * 128;
    static constexpr int SC_BYTES = MODE == MODE_FWD ? BM * 8 : (MODE == MODE_BWD ? 128 : 0);
    static constexpr int STAGE_BYTES = (A_BYTES + B_BYTES + SC_BYTES + 1023) / 1024 * 1024;
};

template <int BM, int BN, int WM, int WN, int STAGES, int MODE, int EPI, int MINB>
__global__ void __launch_bounds__(256, MINB) gemm_tn_dmma(const GemmParams p) {
    constexpr int WGM = BM / WM, WGN = BN / WN;
    static_assert(WGM * WGN == 8, "8 warps per CTA");
    static_assert(WM % 16 == 0 && WN % 16 == 0, "warp tile must hold whole 16-row groups");
    constexpr int FM = WM / 8, FN = WN / 8;
    using TC = TileCfg<BM, BN, MODE>;

    extern __shared__ unsigned char smem_raw[];
    const uint32_t smem_base = (static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)) + 1023u) & ~1023u;
    unsigned char* smem_gen = smem_raw + (smem_base - static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)));

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp % WGM, wn = warp / WGM;
    const int g = lane >> 2, q = lane & 3;
    const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN, z = blockIdx.z;

    int kt0, kt1;
    if (MODE == MODE_BWD) {
        kt0 = 0;
        kt1 = p.kt_total;
    } else {
        kt0 = z * p.kt_per_split;
        kt1 = min(kt0 + p.kt_per_split, p.kt_total);
    }
    const int nkt = max(kt1 - kt0, 0);

    // ---- producer: one k-tile (A BMx16, B BNx16, scale slice) into stage `slot` -------------------
    auto load_stage = [&](int kt, int slot) {
        const uint32_t sA = smem_base + slot * TC::STAGE_BYTES;
        const uint32_t sB = sA + TC::A_BYTES;
        const uint32_t sS = sB + TC::B_BYTES;
        const int64_t a_col = (MODE == MODE_FWD ? (kt % p.a_wrap) : kt) * (int64_t)BK;
        const int64_t b_col = (int64_t)kt * BK;
#pragma unroll
        for (int id = tid; id < BM * 8; id += 256) {
            const int row = id >> 3, ch = id & 7;
            const bool valid = (m0 + row) < p.M;
            const double* src = p.A + (valid ? (int64_t)(m0 + row) * p.lda + a_col + ch * 2 : 0);
            cp_async16(sA + row * 128 + ((ch ^ (row & 7)) << 4), src, valid);
        }
#pragma unroll
        for (int id = tid; id < BN * 8; id += 256) {
            const int row = id >> 3, ch = id & 7;
            const bool valid = (n0 + row) < p.N;
            const double* src = p.B + (valid ? (int64_t)(n0 + row) * p.ldb + b_col + ch * 2 : 0);
            cp_async16(sB + row * 128 + ((ch ^ (row & 7)) << 4), src, valid);
        }
        if (MODE == MODE_FWD) {
            const int v = kt / p.a_wrap;
            if (tid < BM / 2) {
                const bool valid = (m0 + 2 * tid) < p.M;
                const double* src = p.scale + (valid ? (int64_t)v * p.lds + m0 + 2 * tid : 0);
                cp_async16(sS + tid * 16, src, valid);
            }
        } else if (MODE == MODE_BWD) {
            if (tid < 8) cp_async16(sS + tid * 16, p.scale + (int64_t)z * p.lds + b_col + 2 * tid, true);
        }
    };

    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // fragment addressing (doubles): row*16 + (((chunk ^ (row&7)) << 1) | (q&1)), chunk = 2*ks + (q>>1)
    const int xr0 = (2 * (g & 3)), xr1 = xr0 | 1;  // (row & 7) for parity 0 / 1
    int rowA[FM], rowB[FN];
#pragma unroll
    for (int i = 0; i < FM; ++i) rowA[i] = wm * WM + 16 * (i >> 1) + 2 * g + (i & 1);
#pragma unroll
    for (int j = 0; j < FN; ++j) rowB[j] = wn * WN + 16 * (j >> 1) + 2 * g + (j & 1);

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nkt) load_stage(kt0 + s, s);
        cp_async_commit();
    }

    for (int it = 0; it < nkt; ++it) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            const int nx = it + STAGES - 1;
            if (nx < nkt) load_stage(kt0 + nx, nx % STAGES);
            cp_async_commit();
        }
        const int slot = it % STAGES;
        const double* As = reinterpret_cast<const double*>(smem_gen + slot * TC::STAGE_BYTES);
        const double* Bs = reinterpret_cast<const double*>(smem_gen + slot * TC::STAGE_BYTES + TC::A_BYTES);
        const double* Sc =
            reinterpret_cast<const double*>(smem_gen + slot * TC::STAGE_BYTES + TC::A_BYTES + TC::B_BYTES);

        double fv[FM];
        if (MODE == MODE_FWD) {
#pragma unroll
            for (int i = 0; i < FM; ++i) fv[i] = Sc[rowA[i]];
        }
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
            const int ch = 2 * ks + (q >> 1);
            const int c0 = ((ch ^ xr0) << 1) | (q & 1);
            const int c1 = ((ch ^ xr1) << 1) | (q & 1);
            double a[FM], b[FN];
#pragma unroll
            for (int i = 0; i < FM; ++i) a[i] = As[rowA[i] * 16 + ((i & 1) ? c1 : c0)];
#pragma unroll
            for (int j = 0; j < FN; ++j) b[j] = Bs[rowB[j] * 16 + ((j & 1) ? c1 : c0)];
            if (MODE == MODE_FWD) {
#pragma unroll
                for (int i = 0; i < FM; ++i) a[i] *= fv[i];
            } else if (MODE == MODE_BWD) {
                const double sk = Sc[4 * ks + q];
                if (FM <= FN) {
#pragma unroll
                    for (int i = 0; i < FM; ++i) a[i] *= sk;
                } else {
#pragma unroll
                    for (int j = 0; j < FN; ++j) b[j] *= sk;
                }
            }
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma_8x8x4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();
    __syncthreads();

    // ---- epilogue ------------------------------------------------------------------------------
    // acc[i][j][e]: row m = m0 + rowA[i] (i even/odd = adjacent rows), col n = n0 + wn*WN + 16*(j>>1) + 2*(2q+e) + (j&1)
    if (EPI == EPI_STORE) {
        double* outb = p.out + (int64_t)z * p.out_split_stride;
        const bool vec_ok = ((p.ldo & 1) == 0) && ((reinterpret_cast<uintptr_t>(outb) & 15) == 0);
#pragma unroll
        for (int i2 = 0; i2 < FM / 2; ++i2) {
            const int r0 = m0 + wm * WM + 16 * i2 + 2 * g;
#pragma unroll
            for (int j = 0; j < FN; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                    if (n >= p.N) continue;
                    double* ptr = outb + (int64_t)n * p.ldo + r0;
                    const double v0 = acc[2 * i2][j][e], v1 = acc[2 * i2 + 1][j][e];
                    if (vec_ok && r0 + 1 < p.M) {
                        *reinterpret_cast<double2*>(ptr) = make_double2(v0, v1);
                    } else {
                        if (r0 < p.M) ptr[0] = v0;
                        if (r0 + 1 < p.M) ptr[1] = v1;
                    }
                }
        }
    } else {
        const int64_t voff = (int64_t)z * p.n_c;
        const bool vec_ok = ((voff & 1) == 0) && ((p.ldo & 1) == 0) && ((p.ldx & 1) == 0) &&
                            ((reinterpret_cast<uintptr_t>(p.out) & 15) == 0) &&
                            (EPI == EPI_START || (reinterpret_cast<uintptr_t>(p.X) & 15) == 0);
        double part[FN][2];
#pragma unroll
        for (int j = 0; j < FN; ++j) part[j][0] = part[j][1] = 0.0;
#pragma unroll
        for (int i2 = 0; i2 < FM / 2; ++i2) {
            const int r0 = m0 + wm * WM + 16 * i2 + 2 * g;
            if (r0 >= p.M) continue;
            const bool two = (r0 + 1 < p.M);
            const double s0 = p.s[voff + r0], s1 = two ? p.s[voff + r0 + 1] : 0.0;
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
                    const double u0 = acc[2 * i2][j][e], u1 = acc[2 * i2 + 1][j][e];
                    double y0, y1;
                    if (EPI == EPI_CASIDA) {
                        const double* xp = p.X + (int64_t)n * p.ldx + voff + r0;
                        double x0, x1 = 0.0;
                        if (vec_ok && two) {
                            const double2 xv = *reinterpret_cast<const double2*>(xp);
                            x0 = xv.x;
                            x1 = xv.y;
                        } else {
                            x0 = xp[0];
                            if (two) x1 = xp[1];
                        }
                        y0 = d0 * x0 + 2.0 * (s0 * u0);
                        y1 = d1 * x1 + 2.0 * (s1 * u1);
                        part[j][e] += x0 * y0 + x1 * y1;
                    } else {
                        y0 = s0 * u0;
                        y1 = s1 * u1;
                        part[j][e] += y0 * y0 + y1 * y1;
                    }
                    double* yp = p.out + (int64_t)n * p.ldo + voff + r0;
                    if (vec_ok && two) {
                        *reinterpret_cast<double2*>(yp) = make_double2(y0, y1);
                    } else {
                        yp[0] = y0;
                        if (two) yp[1] = y1;
                    }
                }
        }
        if (p.dotpart != nullptr) {
            double* red = reinterpret_cast<double*>(smem_gen);  // [WGM][BN]; the stages are idle now
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
            __syncthreads();
            if (tid < BN && n0 + tid < p.N) {
                double ssum = 0.0;
#pragma unroll
                for (int w = 0; w < WGM; ++w) ssum += red[w * BN + tid];
                p.dotpart[(int64_t)(n0 + tid) * p.dot_stride + (int64_t)z * gridDim.x + blockIdx.x] = ssum;
            }
        }
    }
}

constexpr int kStages = 4;

template <int BM, int BN, int WM, int WN, int MODE, int EPI, int MINB>
cudaError_t launch_one(const GemmParams& p, dim3 grid, cudaStream_t st) {
    using TC = TileCfg<BM, BN, MODE>;
    constexpr int SMEM = kStages * TC::STAGE_BYTES + 1024;
    auto kern = gemm_tn_dmma<BM, BN, WM, WN, kStages, MODE, EPI, MINB>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    kern<<<grid, 256, SMEM, st>>>(p);
    count_launch();
    return cudaGetLastError();
}

template <int MODE, int EPI>
cudaError_t launch_mode(const GemmPlan& plan, const GemmParams& p, int nz, cudaStream_t st) {
    dim3 grid((unsigned)ceil_div(p.M, plan.bm), (unsigned)ceil_div(p.N, plan.bn), (unsigned)nz);
    if (plan.bn == 128) return launch_one<128, 128, 32, 64, MODE, EPI, 1>(p, grid, st);
    return launch_one<128, 64, 32, 32, MODE, EPI, 2>(p, grid, st);
}

}  // namespace

GemmPlan plan_gemm(int mode, int M, int N, int kt_total, int a_wrap, int n_sm) {
    (void)a_wrap;
    GemmPlan pl;
    pl.bm = 128;
    pl.bn = (N > 64) ? 128 : 64;
    pl.splits = 1;
    pl.kt_per_split = kt_total;
    if (mode == MODE_BWD) return pl;
    const int64_t tiles = ceil_div(M, pl.bm) * ceil_div(N, pl.bn);
    const int64_t slots = (int64_t)n_sm * (pl.bn == 64 ? 2 : 1);
    const int min_kt = 8;
    int64_t best_cost = -1;
    int best_s = 1;
    const int max_s = (int)std::max<int64_t>(1, std::min<int64_t>(64, kt_total / min_kt));
    for (int s = 1; s <= max_s; ++s) {
        const int64_t kps = ceil_div(kt_total, s);
        const int64_t real_s = ceil_div(kt_total, kps);
        const int64_t waves = ceil_div(tiles * real_s, slots);
        const int64_t cost = waves * (kps + 6);  // +6 k-tiles: pipeline fill and epilogue of a CTA
        if (best_cost < 0 || cost < best_cost) {
            best_cost = cost;
            best_s = (int)real_s;
        }
    }
    pl.kt_per_split = (int)ceil_div(kt_total, best_s);
    pl.splits = (int)ceil_div(kt_total, pl.kt_per_split);
    return pl;
}

cudaError_t launch_gemm(int mode, int epi, const GemmPlan& plan, const GemmParams& p, int nz, cudaStream_t st) {
    if (p.M <= 0 || p.N <= 0 || nz <= 0) return cudaSuccess;
    if (mode == MODE_FWD && epi == EPI_STORE) return launch_mode<MODE_FWD, EPI_STORE>(plan, p, nz, st);
    if (mode == MODE_PLAIN && epi == EPI_STORE) return launch_mode<MODE_PLAIN, EPI_STORE>(plan, p, nz, st);
    if (mode == MODE_BWD && epi == EPI_CASIDA) return launch_mode<MODE_BWD, EPI_CASIDA>(plan, p, nz, st);
    if (mode == MODE_BWD && epi == EPI_START) return launch_mode<MODE_BWD, EPI_START>(plan, p, nz, st);
    return cudaErrorInvalidValue;
}

}  // namespace gwl
