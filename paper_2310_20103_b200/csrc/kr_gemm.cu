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
#include "kr_gemm_common.cuh"

namespace gwl {

thread_local int64_t* g_launch_counter = nullptr;

namespace {

constexpr int FWD_VCHUNK = 256;  // K.X k-tile order: occupied orbitals per chunk (see the producer loop)
constexpr int BWD_MIN_UNITS = 16;  // fewest k-tiles worth handing to one more CTA

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
    __shared__ double red[(EPI == EPI_STORE) ? 1 : (BM / WM) * BN];  // per-column dot partials of the epilogue
    const uint32_t smem_base = (static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)) + 1023u) & ~1023u;
    unsigned char* smem_gen = smem_raw + (smem_base - static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw)));
    const uint32_t bar_base = static_cast<uint32_t>(__cvta_generic_to_shared(bars));
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp % WGM, wn = (warp / WGM) % WGN;
    const int g = lane >> 2, q = lane & 3;
    // ---- work list ------------------------------------------------------------------------------------
    // FWD / PLAIN: one segment per CTA, (m-tile, n-tile, split) = blockIdx.
    // BWD: a persistent 1-D grid of G CTAs over the tiles, v fastest (tile = (m-tile, n-tile, v)), in two phases.
    //  (1) R = floor(tiles / G) aligned rounds: CTA g takes tile i*G + g whole.  All CTAs walk the same k-range at the
    //      same time and neighbouring CTAs differ only in v, so they read the SAME Phi_c^T and W k-tiles: each comes
    //      from HBM once and is an L2 hit for the others.
    //  (2) the remaining tiles ("stream-K"): their tiles x k-tiles unit space is cut into G equal contiguous ranges,
    //      so a range starts and ends in the middle of a tile.  The CTA whose range holds the LAST k-tile of a tile
    //      owns it (sums the partials of the others in a fixed order and runs the epilogue); the others store their
    //      accumulators to the workspace and raise a flag.  A range is processed head-of-last-tile first and
    //      tail-of-first-tile last: contributions are written at the start of the phase, collected at its end, and an
    //      owner only ever waits for CTAs of LOWER index (dispatched no later than itself).
    const int KT = p.kt_total;
    int ns = 1, nr = 0, ns_tail = 0, first_tile = 0, tile0 = 0, gt = 1;
    int64_t u0 = 0, u1 = 0, U = 0;
    if (MODE == MODE_BWD) {
        nr = p.n_tiles / (int)gridDim.x;
        tile0 = nr * (int)gridDim.x;
        U = (int64_t)(p.n_tiles - tile0) * KT;
        // CTAs sharing phase 2: at least BWD_MIN_UNITS k-tiles each (every cut costs a partial tile through the
        // workspace), never an empty range in front of a non-empty one (an owner waits for ALL lower CTAs of its tile)
        gt = (int)min((int64_t)gridDim.x, max((int64_t)(p.n_tiles - tile0), U / BWD_MIN_UNITS));
        if ((int)blockIdx.x < gt) {
            u0 = U * blockIdx.x / gt;
            u1 = U * (blockIdx.x + 1) / gt;
            first_tile = tile0 + (int)(u0 / KT);
            ns_tail = u1 > u0 ? tile0 + (int)((u1 - 1) / KT) - first_tile + 1 : 0;
        }
        ns = nr + ns_tail;
    }
    auto seg_at = [&](int i, int& tile, int& kb, int& ke) {
        if (MODE != MODE_BWD) {
            tile = 0;
            kb = min(blockIdx.z * p.kt_per_split, KT);
            ke = min(kb + p.kt_per_split, KT);
            return;
        }
        if (i < nr) {
            tile = i * (int)gridDim.x + (int)blockIdx.x;
            kb = 0;
            ke = KT;
            return;
        }
        i -= nr;
        const int sidx = ns_tail == 1 ? 0 : (i == 0 ? ns_tail - 1 : (i == ns_tail - 1 ? 0 : i));
        tile = first_tile + sidx;
        const int64_t tb = (int64_t)(tile - tile0) * KT;
        kb = (int)(max(u0, tb) - tb);
        ke = (int)(min(u1, tb + KT) - tb);
    };
    auto tile_coords = [&](int tile, int& m0, int& n0, int& z) {
        if (MODE != MODE_BWD) {
            m0 = blockIdx.x * BM;
            n0 = blockIdx.y * BN;
            z = blockIdx.z;
        } else {
            // v fastest.  Tried in round 2 and dropped: groups of G v's with the m-tile inside a group (to keep a group's rows of
            // Phi_v^T in L2): 25.8 GB instead of 18.3 GB of DRAM reads per launch at config 4 and 0.6 % slower -- a new 21 MB
            // Phi_c^T slice every round costs more than the Phi_v^T rows it saves.
            z = tile % p.scale_rows;  // v
            const int r = tile / p.scale_rows;
            n0 = (r % p.tiles_n) * BN;
            m0 = (r / p.tiles_n) * BM;
        }
    };

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
    pdl_trigger();
    pdl_wait();  // everything above overlapped the tail of the previous kernel; no global access before this point

    if (warp >= NCW) {
        // ---- producer warpgroup: TMA the k-tiles (A BMx16, B BNx16, scale slice) of each stage ---------------
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;\n");
        if (warp == NCW && lane == 0) {
            int it = 0;
            for (int i = 0; i < ns; ++i) {
                int tile, kb, ke, m0, n0, z;
                seg_at(i, tile, kb, ke);
                tile_coords(tile, m0, n0, z);
                for (int kt = kb; kt < ke; ++kt, ++it) {
                    const int slot = it % STAGES;
                    const uint32_t par = ((it / STAGES) & 1) ^ 1;  // passes at once on a fresh barrier
                    while (!mbar_try_wait(empty_bar(slot), par)) {
                    }
                    const uint32_t fb = full_bar(slot);
                    mbar_expect_tx(fb, TC::TX_BYTES);
                    const uint32_t sA = smem_base + slot * TC::KT_BYTES;
                    const uint32_t sB = sA + TC::A_BYTES;
                    const uint32_t sS = sB + TC::B_BYTES;
                    if (MODE == MODE_FWD) {
                        // k-tile order (chunk of FWD_VCHUNK occupied orbitals, c-tile, v in chunk).  The A tile (Phi_c rows of
                        // this m-tile, 16 columns) is the same for a whole run of v and is an L2 hit, one chunk's row scales
                        // (FWD_VCHUNK x BM doubles = 64 KB) stay in L2 over all c-tiles, and Phi_c is streamed once per chunk.
                        // DRAM reads of one launch at config 4 (ncu): v outermost (round 1) 703 GB -- every CTA re-streamed
                        // its slice of Phi_c once per v --, v innermost 58.7 GB (the row scales once per c-tile), against
                        // about 5 GB algorithmic.  The B tile is xs[:, v, c-tile]: a strided walk over xs, read once either way.
                        const int per_chunk = p.a_wrap * FWD_VCHUNK;
                        const int chunk = kt / per_chunk, rem = kt - chunk * per_chunk;
                        const int vlen = min(FWD_VCHUNK, p.scale_rows - chunk * FWD_VCHUNK);
                        const int ct = rem / vlen, v = chunk * FWD_VCHUNK + (rem - ct * vlen);
                        tma_load_2d(sA, &tmA, ct * BK, m0, fb);
                        tma_load_2d(sB, &tmB, (v * p.a_wrap + ct) * BK, n0, fb);
                        tma_load_2d(sS, &tmS, m0, v, fb);
                    } else {
                        tma_load_2d(sA, &tmA, kt * BK, m0, fb);
                        tma_load_2d(sB, &tmB, kt * BK, n0, fb);
                        if (MODE == MODE_BWD) tma_load_2d(sS, &tmS, kt * BK, z, fb);
                    }
                }
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(CREGS));

    double acc[FM][FN][2];
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
    constexpr bool FV_REGS = (MODE == MODE_FWD) && FN <= 4;
    double fv[FV_REGS ? FM : 1];  // FWD, narrow tiles: phi_v row scales of the k-tile being fetched

    auto fetch = [&](int slot, int ks, double(&a)[FM], double(&b)[FN]) {
        const unsigned char* base = smem_gen + slot * TC::KT_BYTES;
        const double* As = reinterpret_cast<const double*>(base);
        const double* Bs = reinterpret_cast<const double*>(base + TC::A_BYTES);
        const double* Sc = reinterpret_cast<const double*>(base + TC::A_BYTES + TC::B_BYTES);
        const int ch = 2 * ks + (q >> 1);
        const int c0 = ((ch ^ xr0) << 1) | (q & 1);
        const int c1 = ((ch ^ xr1) << 1) | (q & 1);
#pragma unroll
        for (int i = 0; i < FM; ++i) a[i] = As[rowA[i] * 16 + ((i & 1) ? c1 : c0)];
#pragma unroll
        for (int j = 0; j < FN; ++j) b[j] = Bs[rowB[j] * 16 + ((j & 1) ? c1 : c0)];
        if (MODE == MODE_FWD) {
            // wide warp tiles (FN = 8, 232 registers): the row scales are re-read from shared memory at every k-step
            // instead of living in FM registers for the whole k-tile (measured at config 2: K.X 24.0 -> 23.8 ms);
            // narrow ones (FN = 4) have the registers and fewer DMMAs per k-step to hide the extra LDS behind.
            if (FV_REGS) {
                if (ks == 0) {
#pragma unroll
                    for (int i = 0; i < FM; ++i) fv[i] = Sc[rowA[i]];
                }
#pragma unroll
                for (int i = 0; i < FM; ++i) a[i] *= fv[i];
            } else {
#pragma unroll
                for (int i = 0; i < FM; ++i) a[i] *= Sc[rowA[i]];
            }
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

    int it = 0;  // k-tiles consumed so far by this CTA (ring position), continuous across segments
    for (int si = 0; si < ns; ++si) {
        int tile, kb, ke, m0, n0, z;
        seg_at(si, tile, kb, ke);
        tile_coords(tile, m0, n0, z);
        const int nkt = ke - kb;
#pragma unroll
        for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        if (nkt > 0) {
            const int slot = it % STAGES;
            const uint32_t par = (it / STAGES) & 1;
            while (!mbar_try_wait(full_bar(slot), par)) {
            }
            fetch(slot, 0, fa[0], fb[0]);
        }
        for (int j = 0; j < nkt; ++j, ++it) {
            const int slot = it % STAGES;
            const int nslot = (it + 1) % STAGES;
            const uint32_t npar = ((it + 1) / STAGES) & 1;
            const bool has_next = (j + 1 < nkt);
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
            // ---- stream-K hand-over: partial tiles go through the workspace, in accumulator order -------------
            // ws[cta][((warp*FM + i)*FN + j)*2 + e][lane]: every store / load of a warp is one 256-byte row
            constexpr int TILE_ELEMS = NCW * FM * FN * 2 * 32;
            if (ke < KT) {
                double* wsp = p.ws + (int64_t)blockIdx.x * TILE_ELEMS + (int64_t)warp * (FM * FN * 2 * 32) + lane;
#pragma unroll
                for (int i = 0; i < FM; ++i)
#pragma unroll
                    for (int j = 0; j < FN; ++j)
#pragma unroll
                        for (int e = 0; e < 2; ++e) wsp[((i * FN + j) * 2 + e) * 32] = acc[i][j][e];
                asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");
                if (tid == 0) {
                    __threadfence();
                    asm volatile("st.release.gpu.global.u32 [%0], %1;\n" ::"l"(p.flags + blockIdx.x), "r"(p.epoch) : "memory");
                }
                continue;
            }
            if (kb > 0) {
                const int64_t tb = (int64_t)(tile - tile0) * KT;
                int gf = blockIdx.x;  // first contributor: the CTA whose range holds the tile's first k-tile
                while (gf > 0 && U * gf / gt > tb) --gf;
                if (tid == 0) {
                    for (int c = gf; c < (int)blockIdx.x; ++c) {
                        unsigned f;
                        do {
                            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(f) : "l"(p.flags + c) : "memory");
                        } while (f != p.epoch);
                    }
                }
                asm volatile("bar.sync 1, %0;\n" ::"n"(NCW * 32) : "memory");
                for (int c = gf; c < (int)blockIdx.x; ++c) {
                    const double* wsp = p.ws + (int64_t)c * TILE_ELEMS + (int64_t)warp * (FM * FN * 2 * 32) + lane;
#pragma unroll
                    for (int i = 0; i < FM; ++i)
#pragma unroll
                        for (int j = 0; j < FN; ++j)
#pragma unroll
                            for (int e = 0; e < 2; ++e) acc[i][j][e] += __ldcg(wsp + ((i * FN + j) * 2 + e) * 32);
                }
            }
            const int64_t voff = (int64_t)z * p.n_c;
            if (EPI == EPI_CHEB) {
                // ---- one Chebyshev term of p_g(C): t = ca (C x) + cb x + cc t0, w += cw t, xs = s o t, dots q.w -------
                const bool vec2 = ((voff & 1) == 0) && ((p.ldx & 1) == 0) &&
                                  (((reinterpret_cast<uintptr_t>(p.X) | reinterpret_cast<uintptr_t>(p.out) |
                                     reinterpret_cast<uintptr_t>(p.Wacc) | reinterpret_cast<uintptr_t>(p.T0) |
                                     reinterpret_cast<uintptr_t>(p.Q)) & 15) == 0);
                const bool has_t0 = p.T0 != nullptr, has_q = p.Q != nullptr, first = p.first != 0;
                const double cpl = p.coupling, ca = p.ca, cb = p.cb, cc = p.cc, cw = p.cw, c0 = p.c0;
                double part[FN][2];
#pragma unroll
                for (int j = 0; j < FN; ++j) part[j][0] = part[j][1] = 0.0;
                auto ld2 = [&](const double* ptr, bool two, double& a, double& b) {
                    if (vec2 && two) {
                        const double2 v2 = *reinterpret_cast<const double2*>(ptr);
                        a = v2.x;
                        b = v2.y;
                    } else {
                        a = ptr[0];
                        b = two ? ptr[1] : 0.0;
                    }
                };
                auto st2 = [&](double* ptr, bool two, double a, double b) {
                    if (vec2 && two) {
                        *reinterpret_cast<double2*>(ptr) = make_double2(a, b);
                    } else {
                        ptr[0] = a;
                        if (two) ptr[1] = b;
                    }
                };
#pragma unroll
                for (int i2 = 0; i2 < FM / 2; ++i2) {
                    const int r0 = m0 + wm * WM + 16 * i2 + 2 * g;
                    if (r0 >= p.M) continue;
                    const bool two = (r0 + 1 < p.M);
                    const double s0 = p.s[voff + r0], s1 = two ? p.s[voff + r0 + 1] : 0.0;
                    const double d0 = p.d2[voff + r0], d1 = two ? p.d2[voff + r0 + 1] : 0.0;
                    constexpr int JB = 2;  // columns whose loads are in flight together (3-4 streams of 16 bytes each)
#pragma unroll
                    for (int j0 = 0; j0 < FN; j0 += JB) {
                        double xr[JB][2][2], tr[JB][2][2], wr[JB][2][2], qr[JB][2][2];
#pragma unroll
                        for (int jj = 0; jj < JB; ++jj)
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int j = j0 + jj;
                                const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                                xr[jj][e][0] = xr[jj][e][1] = tr[jj][e][0] = tr[jj][e][1] = 0.0;
                                wr[jj][e][0] = wr[jj][e][1] = qr[jj][e][0] = qr[jj][e][1] = 0.0;
                                if (n >= p.N) continue;
                                const int64_t off = (int64_t)n * p.ldx + voff + r0;
                                ld2(p.X + off, two, xr[jj][e][0], xr[jj][e][1]);
                                if (has_t0) ld2(p.T0 + off, two, tr[jj][e][0], tr[jj][e][1]);
                                if (!first) ld2(p.Wacc + off, two, wr[jj][e][0], wr[jj][e][1]);
                                if (has_q) ld2(p.Q + off, two, qr[jj][e][0], qr[jj][e][1]);
                            }
#pragma unroll
                        for (int jj = 0; jj < JB; ++jj)
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int j = j0 + jj;
                                const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                                if (n >= p.N) continue;
                                const double x0 = xr[jj][e][0], x1 = xr[jj][e][1];
                                const double y0 = d0 * x0 + cpl * (s0 * acc[2 * i2][j][e]);
                                const double y1 = d1 * x1 + cpl * (s1 * acc[2 * i2 + 1][j][e]);
                                double t0v = ca * y0 + cb * x0, t1v = ca * y1 + cb * x1;
                                if (has_t0) {
                                    t0v += cc * tr[jj][e][0];
                                    t1v += cc * tr[jj][e][1];
                                }
                                const double w0 = first ? c0 * x0 + cw * t0v : wr[jj][e][0] + cw * t0v;
                                const double w1 = first ? c0 * x1 + cw * t1v : wr[jj][e][1] + cw * t1v;
                                const int64_t off = (int64_t)n * p.ldx + voff + r0;
                                st2(p.Wacc + off, two, w0, w1);
                                if (p.xs_out != nullptr) {  // not the last term: t and its scaled copy feed the next one
                                    st2(p.out + off, two, t0v, t1v);
                                    // n_cp is a multiple of 16 and r0 is even: always 16-byte aligned
                                    double* xp = p.xs_out + (int64_t)n * p.ldxs + (int64_t)z * p.n_cp + r0;
                                    if (two) {
                                        *reinterpret_cast<double2*>(xp) = make_double2(s0 * t0v, s1 * t1v);
                                    } else {
                                        xp[0] = s0 * t0v;
                                    }
                                }
                                if (has_q) part[j][e] += qr[jj][e][0] * w0 + qr[jj][e][1] * w1;
                            }
                    }
                }
                if (p.dotpart != nullptr && has_q) {
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
                        p.dotpart[(int64_t)(n0 + tid) * p.dot_stride + (int64_t)z * p.tiles_m + m0 / BM] = ssum;
                    }
                }
                continue;
            }
            const bool vec_ok = ((voff & 1) == 0) && ((p.ldo & 1) == 0) && ((p.ldx & 1) == 0) &&
                                ((reinterpret_cast<uintptr_t>(p.out) & 15) == 0) &&
                                (EPI == EPI_START || (reinterpret_cast<uintptr_t>(p.X) & 15) == 0);
            const double cpl = p.coupling;
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
                // the x loads of a batch of JB columns are issued before its first store: one L2 round trip per batch
                // instead of one per element (x and out never alias, include/gwl.h, but the compiler cannot know);
                // wide warp tiles take two batches so that the batch fits beside the 128 accumulator registers
                constexpr int JB = FN > 4 ? FN / 2 : FN;
#pragma unroll
                for (int j0 = 0; j0 < FN; j0 += JB) {
                    double xr[JB][2][2];
                    if (EPI == EPI_CASIDA) {
#pragma unroll
                        for (int jj = 0; jj < JB; ++jj)
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int j = j0 + jj;
                                const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                                xr[jj][e][0] = xr[jj][e][1] = 0.0;
                                if (n >= p.N) continue;
                                const double* xp = p.X + (int64_t)n * p.ldx + voff + r0;
                                if (vec_ok && two) {
                                    const double2 xv = __ldg(reinterpret_cast<const double2*>(xp));
                                    xr[jj][e][0] = xv.x;
                                    xr[jj][e][1] = xv.y;
                                } else {
                                    xr[jj][e][0] = __ldg(xp);
                                    if (two) xr[jj][e][1] = __ldg(xp + 1);
                                }
                            }
                    }
#pragma unroll
                    for (int jj = 0; jj < JB; ++jj)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int j = j0 + jj;
                            const int n = n0 + wn * WN + 16 * (j >> 1) + 2 * (2 * q + e) + (j & 1);
                            if (n >= p.N) continue;
                            const double u0v = acc[2 * i2][j][e], u1v = acc[2 * i2 + 1][j][e];
                            double y0, y1;
                            if (EPI == EPI_CASIDA) {
                                const double x0 = xr[jj][e][0], x1 = xr[jj][e][1];
                                y0 = d0 * x0 + cpl * (s0 * u0v);
                                y1 = d1 * x1 + cpl * (s1 * u1v);
                                part[j][e] += x0 * y0 + x1 * y1;
                            } else {
                                y0 = s0 * u0v;
                                y1 = s1 * u1v;
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
                // the producer is already refilling the stage ring for the next tile: `red` is its own array
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
                    p.dotpart[(int64_t)(n0 + tid) * p.dot_stride + (int64_t)z * p.tiles_m + m0 / BM] = ssum;
                }
            }
        }
    }
}

template <int BM, int BN, int WM, int WN, int STAGES, int MODE, int EPI, int CREGS>
cudaError_t launch_one(const GemmParams& p, dim3 grid, cudaStream_t st) {
    using TC = TileCfg<BM, BN, MODE>;
    constexpr int SMEM = STAGES * TC::KT_BYTES + 1024;
    constexpr int NTHREADS = ((BM / WM) * (BN / WN) + 4) * 32;
    static_assert(SMEM <= 227 * 1024, "stage ring does not fit in shared memory");
    auto kern = gemm_tn_dmma<BM, BN, WM, WN, STAGES, MODE, EPI, CREGS>;
    static SmemAttr attr;  // per device (the attribute is a property of the function ON a device)
    cudaError_t ea = attr.ensure(kern, SMEM);
    if (ea != cudaSuccess) return ea;
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
    cudaError_t le = launch_pdl(kern, grid, dim3(NTHREADS), SMEM, st, 1u, p, tmA, tmB, tmS);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

// BWD grid: one CTA per SM, fewer only when the whole product has too few k-tiles to be worth cutting
// (every cut costs one partial tile through the workspace).
int bwd_grid(int64_t tiles, int kt_total, int n_sm) {
    const int64_t by_units = tiles * kt_total / BWD_MIN_UNITS;
    return (int)std::max<int64_t>(1, std::min<int64_t>(n_sm, std::max<int64_t>(std::min<int64_t>(tiles, n_sm), by_units)));
}

template <int MODE, int EPI>
cudaError_t launch_mode(const GemmPlan& plan, const GemmParams& p0, int nz, cudaStream_t st) {
    GemmParams p = p0;
    p.tiles_m = (int)ceil_div(p.M, plan.bm);
    p.tiles_n = (int)ceil_div(p.N, plan.bn);
    p.n_tiles = p.tiles_m * p.tiles_n * nz;
    dim3 grid((unsigned)p.tiles_m, (unsigned)p.tiles_n, (unsigned)nz);
    if (MODE == MODE_BWD) {
        if (p.ws == nullptr || p.flags == nullptr || p.epoch == 0 || p.n_sm <= 0) return cudaErrorInvalidValue;
        grid = dim3((unsigned)bwd_grid(p.n_tiles, p.kt_total, p.n_sm), 1, 1);
    }
    // bn = 128: wide blocks (configs 2-4); bn = 64: narrow blocks (configs 0-1).  Other warp tilings were measured in
    // round 1 (16 consumer warps of 32x32 / 32x16, 64x32 warp tiles, 6- and 8-stage rings) and were slower.
    if (plan.bn == 128) return launch_one<128, 128, 32, 64, 4, MODE, EPI, 232>(p, grid, st);
    return launch_one<128, 64, 32, 32, 4, MODE, EPI, 168>(p, grid, st);
}

}  // namespace

size_t gemm_bwd_ws_bytes(int n_sm) { return (size_t)n_sm * 128 * 128 * sizeof(double); }
size_t gemm_bwd_flag_bytes(int n_sm) { return (size_t)n_sm * sizeof(unsigned); }

GemmPlan plan_gemm(int mode, int M, int N, int kt_total, int a_wrap, int n_sm) {
    (void)a_wrap;
    GemmPlan pl;
    pl.bm = 128;
    pl.bn = (N > 64) ? 128 : 64;  // a 256x64 tile was measured too (config 1): no faster in K.X, slower hand-over in K^T.W
    pl.splits = 1;
    pl.kt_per_split = kt_total;
    if (mode == MODE_BWD) return pl;
    const int64_t tiles = ceil_div(M, pl.bm) * ceil_div(N, pl.bn);
    const int64_t slots = n_sm;  // one CTA per SM (register file)
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
    if (mode == MODE_BWD && epi == EPI_CHEB) return launch_mode<MODE_BWD, EPI_CHEB>(plan, p, nz, st);
    return cudaErrorInvalidValue;
}

}  // namespace gwl
