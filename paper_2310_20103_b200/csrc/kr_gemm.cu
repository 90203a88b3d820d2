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
#include <cuda.h>

#include <cstdlib>

#include "gwl_internal.h"

namespace gwl {

thread_local int64_t* g_launch_counter = nullptr;

#ifdef GWL_TRACE
// Development builds only (-DGWL_TRACE): per-CTA %globaltimer stamps at entry / first tile landed / main loop done /
// epilogue done, 4 x uint64 per CTA, written to a caller-provided device buffer.
unsigned long long* g_trace_buf = nullptr;
extern "C" void gwl_debug_set_trace(unsigned long long* dev_buf) { g_trace_buf = dev_buf; }
#define GWL_STAMP(slot)                                                                            \
    do {                                                                                           \
        if (p.trace != nullptr && (tid & 31) == 0 && warp == 0) {                                  \
            unsigned long long t__;                                                                \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t__));                                \
            p.trace[4 * ((blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) + slot] = t__; \
        }                                                                                          \
    } while (0)
#else
#define GWL_STAMP(slot) \
    do {                \
    } while (0)
#endif

namespace {

// ---- TMA / mbarrier primitives (sm_90+ PTX; SASS: UTMALDG, SYNCS) ---------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];\n" ::"l"(map) : "memory");
}

__device__ __forceinline__ void dmma_8x8x4(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

template <int BM, int BN, int MODE>
struct TileCfg {
    static constexpr int A_BYTES = BM * 128;
    static constexpr int B_BYTES = BN * 128;
    static constexpr int SC_BYTES = MODE == MODE_FWD ? BM * 8 : (MODE == MODE_BWD ? 128 : 0);
    static constexpr int TX_BYTES = A_BYTES + B_BYTES + SC_BYTES;           // one k-tile (16 doubles deep)
    static constexpr int KT_BYTES = (TX_BYTES + 1023) / 1024 * 1024;        // its shared-memory footprint
};

// One CTA = NCW consumer warps (DMMA) + one producer warpgroup (TMA, a single elected lane; the warpgroup gives
// its registers back with setmaxnreg.dec so that the consumers can take CREGS each with setmaxnreg.inc -- the
// register file is per SMSP, so a ninth full-size warp would cap everybody at 168 registers).  A pipeline
// stage holds one k-tile and has one "full" mbarrier (TMA complete_tx) and one "empty" mbarrier
// (one arrive per consumer warp).  There is no CTA-wide barrier in the main loop: consumer warps drift up to
// STAGES-1 stages apart and the producer blocks only on the empty barrier of the slot it refills.
template <int BM, int BN, int WM, int WN, int STAGES, int MODE, int EPI, int CREGS>
__global__ void __launch_bounds__(((BM / WM) * (BN / WN) + 4) * 32, 1)
    gemm_tn_dmma(const GemmParams p, const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                 const __grid_constant__ CUtensorMap tmS) {
    constexpr int WGM = BM / WM, WGN = BN / WN;
    constexpr int NCW = WGM * WGN;
    static_assert(WM % 16 == 0 && WN % 16 == 0, "warp tile must hold whole 16-row groups");
    constexpr int FM = WM / 8, FN = WN / 8;
    using TC = TileCfg<BM, BN, MODE>;

    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[2 * STAGES];
    const uint32_t smem_base = (static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)) + 1023u) & ~1023u;
    unsigned char* smem_gen = smem_raw + (smem_base - static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)));
    const uint32_t bar_base = static_cast<uint32_t>(__cvta_generic_to_shared(bars));
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp % WGM, wn = (warp / WGM) % WGN;
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
    GWL_STAMP(0);

    if (tid == 0) {
        tma_prefetch_desc(&tmA);
        tma_prefetch_desc(&tmB);
        if (MODE != MODE_PLAIN) tma_prefetch_desc(&tmS);
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), NCW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    if (warp >= NCW) {
        // ---- producer warpgroup: TMA the k-tiles (A BMx16, B BNx16, scale slice) of each stage ---------------
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
        if (warp == NCW && lane == 0) {
            for (int it = 0; it < nkt; ++it) {
                const int slot = it % STAGES;
                const uint32_t par = ((it / STAGES) & 1) ^ 1;  // passes at once on a fresh barrier
                while (!mbar_try_wait(empty_bar(slot), par)) {
                }
                const int kt = kt0 + it;
                const uint32_t fb = full_bar(slot);
                mbar_expect_tx(fb, TC::TX_BYTES);
                const uint32_t sA = smem_base + slot * TC::KT_BYTES;
                const uint32_t sB = sA + TC::A_BYTES;
                const uint32_t sS = sB + TC::B_BYTES;
                const int a_col = (MODE == MODE_FWD ? (kt % p.a_wrap) : kt) * BK;
                tma_load_2d(sA, &tmA, a_col, m0, fb);
                tma_load_2d(sB, &tmB, kt * BK, n0, fb);
                if (MODE == MODE_FWD)
                    tma_load_2d(sS, &tmS, m0, kt / p.a_wrap, fb);
                else if (MODE == MODE_BWD)
                    tma_load_2d(sS, &tmS, kt * BK, z, fb);
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(CREGS));

    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    // ---- consumer warps --------------------------------------------------------------------------------
    // fragment addressing (doubles): row*16 + (((chunk ^ (row&7)) << 1) | (q&1)), chunk = 2*ks + (q>>1)
    const int xr0 = (2 * (g & 3)), xr1 = xr0 | 1;  // (row & 7) for parity 0 / 1
    int rowA[FM], rowB[FN];
#pragma unroll
    for (int i = 0; i < FM; ++i) rowA[i] = wm * WM + 16 * (i >> 1) + 2 * g + (i & 1);
#pragma unroll
    for (int j = 0; j < FN; ++j) rowB[j] = wn * WN + 16 * (j >> 1) + 2 * g + (j & 1);

    // The k-steps of all k-tiles form one software pipeline: while the 32 (FM*FN) DMMAs of k-step s issue, the
    // fragments of k-step s+1 are fetched from shared memory and scaled -- across k-tile boundaries too, where
    // the wait on the next "full" barrier is issued one k-step early so that its latency is hidden as well.
    double fa[2][FM], fb[2][FN];  // fragment double buffer, indexed by ks & 1 (all indices are compile-time)
    double fv[FM];                // FWD: phi_v row scales of the k-tile being fetched

    auto fetch = [&](int slot, int ks, double(&a)[FM], double(&b)[FN]) {
        const unsigned char* base = smem_gen + slot * TC::KT_BYTES;
        const double* As = reinterpret_cast<const double*>(base);
        const double* Bs = reinterpret_cast<const double*>(base + TC::A_BYTES);
        const double* Sc = reinterpret_cast<const double*>(base + TC::A_BYTES + TC::B_BYTES);
        if (MODE == MODE_FWD && ks == 0) {
#pragma unroll
            for (int i = 0; i < FM; ++i) fv[i] = Sc[rowA[i]];
        }
        const int ch = 2 * ks + (q >> 1);
        const int c0 = ((ch ^ xr0) << 1) | (q & 1);
        const int c1 = ((ch ^ xr1) << 1) | (q & 1);
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
    };
    auto mma_step = [&](const double(&a)[FM], const double(&b)[FN]) {
#pragma unroll
        for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j) dmma_8x8x4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    };

    if (nkt > 0) {
        while (!mbar_try_wait(full_bar(0), 0)) {
        }
        fetch(0, 0, fa[0], fb[0]);
    }
    GWL_STAMP(1);
    for (int it = 0; it < nkt; ++it) {
        const int slot = it % STAGES;
        const int nslot = (it + 1) % STAGES;
        const uint32_t npar = ((it + 1) / STAGES) & 1;
        const bool has_next = (it + 1 < nkt);
        fetch(slot, 1, fa[1], fb[1]);
        mma_step(fa[0], fb[0]);
        fetch(slot, 2, fa[0], fb[0]);
        mma_step(fa[1], fb[1]);
        bool ready = true;
        if (has_next) ready = mbar_try_wait(full_bar(nslot), npar);  // result is needed one k-step later
        fetch(slot, 3, fa[1], fb[1]);
        mma_step(fa[0], fb[0]);
        if (has_next) {
            while (!ready) ready = mbar_try_wait(full_bar(nslot), npar);
            fetch(nslot, 0, fa[0], fb[0]);
        }
        mma_step(fa[1], fb[1]);
        // every fragment of this k-tile has been consumed by a DMMA: hand the slot back to the producer
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar(slot));
    }

    GWL_STAMP(2);
    // ---- epilogue ------------------------------------------------------------------------------
    // acc[i][j][e]: row m = m0 + rowA[i] (i even/odd = adjacent rows), col n = n0 + wn*WN + 16*(j>>1) + 2*(2q+e) + (j&1)
    constexpr bool consumer = true;  // the producer warpgroup has returned
    if (EPI == EPI_STORE) {
        if (consumer) {
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
        }
    } else {
        const int64_t voff = (int64_t)z * p.n_c;
        const bool vec_ok = ((voff & 1) == 0) && ((p.ldo & 1) == 0) && ((p.ldx & 1) == 0) &&
                            ((reinterpret_cast<uintptr_t>(p.out) & 15) == 0) &&
                            (EPI == EPI_START || (reinterpret_cast<uintptr_t>(p.X) & 15) == 0);
        double part[FN][2];
#pragma unroll
        for (int j = 0; j < FN; ++j) part[j][0] = part[j][1] = 0.0;
        if (consumer) {
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
                // all x loads of this row pair are issued before the first store: one L2 round trip per i2 instead of
                // one per element (x and out never alias, include/gwl.h, but the compiler cannot know)
                double xr[FN][2][2];
                if (EPI == EPI_CASIDA) {
#pragma unroll
                    for (int j = 0; j < FN; ++j)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                            xr[j][e][0] = xr[j][e][1] = 0.0;
                            if (n >= p.N) continue;
                            const double* xp = p.X + (int64_t)n * p.ldx + voff + r0;
                            if (vec_ok && two) {
                                const double2 xv = __ldg(reinterpret_cast<const double2*>(xp));
                                xr[j][e][0] = xv.x;
                                xr[j][e][1] = xv.y;
                            } else {
                                xr[j][e][0] = __ldg(xp);
                                if (two) xr[j][e][1] = __ldg(xp + 1);
                            }
                        }
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
                            const double x0 = xr[j][e][0], x1 = xr[j][e][1];
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
        }
        if (p.dotpart != nullptr) {
            // every TMA write was consumed before the last empty-arrive; the stages can be reused as scratch
            asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");
            double* red = reinterpret_cast<double*>(smem_gen);  // [WGM][BN]
            if (consumer) {
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
    GWL_STAMP(3);
}

using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                             const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                             CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point: libgwl.so has no link-time dependency on libcuda.
EncodeFn get_encode_fn() {
    static EncodeFn fn = nullptr;
    if (fn == nullptr) {
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeFn>(ptr);
    }
    return fn;
}

// 2-D FP64 tensor map over a row-major [rows][ld] array of which `cols` columns are valid; out-of-bounds
// elements of a box read as zero.
cudaError_t make_map(CUtensorMap* m, const double* base, uint64_t cols, uint64_t rows, uint64_t ld, uint32_t box_cols,
                     uint32_t box_rows, bool swizzle) {
    EncodeFn enc = get_encode_fn();
    if (enc == nullptr) return cudaErrorNotSupported;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {ld * sizeof(double)};
    cuuint32_t box[2] = {box_cols, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int BM, int BN, int WM, int WN, int STAGES, int MODE, int EPI, int CREGS>
cudaError_t launch_one(const GemmParams& p, dim3 grid, cudaStream_t st) {
    using TC = TileCfg<BM, BN, MODE>;
    constexpr int SMEM = STAGES * TC::KT_BYTES + 1024;
    constexpr int NTHREADS = ((BM / WM) * (BN / WN) + 4) * 32;
    static_assert(SMEM <= 227 * 1024, "stage ring does not fit in shared memory");
    auto kern = gemm_tn_dmma<BM, BN, WM, WN, STAGES, MODE, EPI, CREGS>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    CUtensorMap tmA, tmB, tmS;
    const uint64_t kcols = (uint64_t)p.kt_total * BK;
    const uint64_t a_cols = MODE == MODE_FWD ? (uint64_t)p.a_wrap * BK : kcols;
    cudaError_t e = make_map(&tmA, p.A, a_cols, (uint64_t)p.M, (uint64_t)p.lda, BK, BM, true);
    if (e != cudaSuccess) return e;
    e = make_map(&tmB, p.B, kcols, (uint64_t)p.N, (uint64_t)p.ldb, BK, BN, true);
    if (e != cudaSuccess) return e;
    if (MODE == MODE_FWD)  // Phi_v^T [n_v][lds]: box = BM row-scale values of one v
        e = make_map(&tmS, p.scale, (uint64_t)p.lds, (uint64_t)p.scale_rows, (uint64_t)p.lds, BM, 1, false);
    else if (MODE == MODE_BWD)  // box = the 16 k-scale values of one v
        e = make_map(&tmS, p.scale, (uint64_t)p.lds, (uint64_t)p.scale_rows, (uint64_t)p.lds, BK, 1, false);
    else
        tmS = tmA;
    if (e != cudaSuccess) return e;
#ifdef GWL_TRACE
    GemmParams pt = p;
    pt.trace = g_trace_buf;
    if (g_trace_buf != nullptr) g_trace_buf += 4ull * grid.x * grid.y * grid.z;  // consecutive launches, consecutive records
    kern<<<grid, NTHREADS, SMEM, st>>>(pt, tmA, tmB, tmS);
#else
    kern<<<grid, NTHREADS, SMEM, st>>>(p, tmA, tmB, tmS);
#endif
    count_launch();
    return cudaGetLastError();
}

// Tile variants.  bn = 128: wide blocks (configs 2-4); bn = 64: narrow blocks (configs 0-1).
// GWL_GEMM_VARIANT (development knob, read once) selects alternative instantiations for sweeps.
int gemm_variant() {
    static int v = -1;
    if (v < 0) {
        const char* e = getenv("GWL_GEMM_VARIANT");
        v = e ? atoi(e) : 0;
    }
    return v;
}

template <int MODE, int EPI>
cudaError_t launch_mode(const GemmPlan& plan, const GemmParams& p, int nz, cudaStream_t st) {
    dim3 grid((unsigned)ceil_div(p.M, plan.bm), (unsigned)ceil_div(p.N, plan.bn), (unsigned)nz);
    const int var = gemm_variant();
    if (plan.bn == 128) {
        switch (var) {
            case 1: return launch_one<128, 128, 32, 32, 4, MODE, EPI, 104>(p, grid, st);  // 16 consumer warps
            case 2: return launch_one<128, 128, 32, 64, 6, MODE, EPI, 232>(p, grid, st);
            case 3: return launch_one<128, 128, 64, 32, 4, MODE, EPI, 232>(p, grid, st);
            default: return launch_one<128, 128, 32, 64, 4, MODE, EPI, 232>(p, grid, st);
        }
    }
    switch (var) {
        case 1: return launch_one<128, 64, 32, 16, 4, MODE, EPI, 104>(p, grid, st);  // 16 consumer warps
        case 2: return launch_one<128, 64, 32, 32, 8, MODE, EPI, 168>(p, grid, st);
        case 3: return launch_one<128, 64, 16, 64, 4, MODE, EPI, 168>(p, grid, st);
        default: return launch_one<128, 64, 32, 32, 4, MODE, EPI, 168>(p, grid, st);
    }
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
