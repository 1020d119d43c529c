// The two dense contractions of the EMC iteration on the 5th-generation tensor cores:
//
//   log-likelihood (north_star stage 2; E-step numerator):
//        L[r,d]  = sum_p logW[r,p] K[d,p] - S[r]         M = R, N = patterns, K-dim = pixels
//   update (eq. 2.5 / 2.11):
//        W'[r,p] = sum_d P[r,d] K[d,p] / s[r]            M = R, N = pixels,   K-dim = patterns
//
// Both are "plane GEMMs": the real-valued operand A (logW or P) is a sum of n_planes 16-bit
// planes (hi + lo); the count operand B is exact in ONE 16-bit plane, so every product is
// exact in fp32 and the only rounding is the fp32 accumulation in TMEM:
//
//        acc[m,n] = sum_pl sum_k A[pl][m][k] * B[n][k]
//
// Kernels: persistent, warp-specialised.
//   warp 0 lane 0 : TMA producer  (cp.async.bulk.tensor -> 128B-swizzled smem ring, mbarrier tx)
//   warp 1 lane 0 : MMA issuer    (tcgen05.mma.kind::f16, fp32 accumulators in TMEM)
//   warps 2..9    : epilogue      (tcgen05.ld 32x32b -> fp32 register accumulators -> fused row op -> out)
// TMEM holds two accumulator stages of BN columns; the K loop alternates between them in chunks
// of 512 elements so that the long sums are carried in round-to-nearest fp32 registers (tcgen05
// accumulation truncates), and the drain of chunk i overlaps the MMAs of chunk i+1.
//   plane_gemm_pair_kernel : the product path.  One CTA PAIR per 256 x BN tile (cta_group::2), results leave
//                            through swizzled staging tiles and TMA stores, the log-likelihood variant also writes
//                            the normalisation's column statistics (tile_out).
//   plane_gemm_kernel      : one CTA per 128 x BN tile (cta_group::1), per-lane stores; EMC_GEMM_1CTA, a
//                            comparison / bisecting aid.
//   simt_plane_gemm_kernel : plain CUDA cores; EMC_DEBUG_SIMT.
#include "emc_internal.cuh"

namespace emc {

namespace {

constexpr int BLOCK_M = 128;
constexpr int BLOCK_K = 64;                    // 64 x 2 B = one 128-byte swizzle row
constexpr int UMMA_K = 16;
constexpr int A_PLANE_BYTES = BLOCK_M * BLOCK_K * 2;
constexpr int kGemmThreads = 320;             // TMA warp, MMA warp, 8 epilogue warps
constexpr int kNumEpiWarps = 8;
constexpr int kChunkKBlocks = 8;               // 8 x 64 = 512 K elements per TMEM accumulation chunk
constexpr int kGroupM = 8;                     // tile rasterisation: 8 m-blocks share each n sweep

template <int NP, int BN, int STAGES>
struct Cfg {
    static constexpr int B_BYTES = BN * BLOCK_K * 2;
    static constexpr int STAGE_BYTES = NP * A_PLANE_BYTES + B_BYTES;
    static constexpr int BAR_BYTES = 256;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + 1024;   // + alignment slack
    static_assert(SMEM_BYTES <= 232448, "exceeds the 227 KB of shared memory per CTA");
    static_assert(2 * BN <= 512, "two accumulator stages must fit the 512 TMEM columns");
    static_assert(BN % 16 == 0 && BN >= 16 && BN <= 256, "UMMA N for M = 128");
    static_assert(BN % 64 == 0, "two epilogue warps per lane quarter read 32 columns at a time");
};

struct GemmArgs {
    int M, N, K;
    int num_m_tiles, num_n_tiles, num_k_blocks;
    float *out;
    int ld_out;
    const float *rowv;
    int epilogue;
    int vec_ok;          // out rows are 16-byte aligned
    int tma_out;         // pair kernel: results leave through the output tensor map (needs vec_ok)
    int k_chunk;         // k-blocks per TMEM accumulation chunk
    const float *chunk_scale;   // [num_chunks][M] factor applied to a chunk when it is drained, or null
    uint32_t idesc;
    // fused column statistics of the log-likelihood epilogue (pair kernel, STATS = true), see tile_out()
    float *stat_m, *stat_w, *stat_z;   // [ceil(M/32)][ld_stat]: reference pair (L, log w) and sum
    int ld_stat;
    const float *weight;        // [M] prior weights w_r or null = uniform
    float log_uniform;          // log(1/R) for weight == null (R = all rotations of the problem, not of this launch)
};

// Gaussian model (EPI_GAUSS, STATS = 2): out = B = acc; the statistics are taken of Q = (B^2 / A_d - C_r) / (2 sigma^2).
// A kernel parameter of its own so that the other instantiations keep their exact parameter block and code.
struct GaussParams {
    const float *g;             // [N] g_d = 1 / (2 sigma^2 A_d), 0 where A_d = 0
    float inv2s2;               // 1 / (2 sigma^2)
};
struct NoGauss {};
template <int STATS> struct GaussOf { typedef NoGauss type; };
template <> struct GaussOf<2> { typedef GaussParams type; };

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrives on the mbarrier once every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t addr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(addr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// UMMA shared-memory descriptor of a K-major tile with 128-byte rows under SWIZZLE_128B:
// start address >> 4 in bits [0,14), LBO (unused for swizzled K-major) = 1 in [16,30),
// SBO = 1024 B (8 rows x 128 B) >> 4 in [32,46), version 1 in [46,48), layout SWIZZLE_128B = 2 in [61,64).
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) |
           (1ull << 46) | (2ull << 61);
}

__device__ __forceinline__ void tile_coords(int tile, const GemmArgs &a, int &m_blk, int &n_blk) {
    const int per_group = kGroupM * a.num_n_tiles;
    const int group = tile / per_group;
    const int first_m = group * kGroupM;
    const int gm = min(a.num_m_tiles - first_m, kGroupM);
    const int t = tile - group * per_group;
    m_blk = first_m + t % gm;
    n_blk = t / gm;
}

// Fused row operation + store of one accumulator row (CW columns starting at column n_base).
template <int CW>
__device__ __forceinline__ void store_row(const float (&racc)[CW], const GemmArgs &args, int m, int n_base, float rv) {
    float *orow = args.out + (size_t)m * args.ld_out;
    // one reciprocal per row (subnormal numerators make a per-element division take its slow path, see tile_out)
    const float inv = rv > 0.f ? 1.f / rv : 0.f;
    const bool inv_ok = !(rv > 0.f) || inv < 3.0e38f;
#pragma unroll
    for (int c = 0; c < CW; c += 4) {
        const int n0 = n_base + c;
        if (n0 >= args.N) break;
        float f[4] = {racc[c], racc[c + 1], racc[c + 2], racc[c + 3]};
        if (args.epilogue == EPI_SUB_ROW) {
#pragma unroll
            for (int j = 0; j < 4; ++j) f[j] -= rv;
        } else if (args.epilogue == EPI_DIV_ROW) {
#pragma unroll
            for (int j = 0; j < 4; ++j) f[j] = inv_ok ? f[j] * inv : (rv > 0.f ? f[j] / rv : 0.f);
        }
        float *o = orow + n0;
        if (args.vec_ok && n0 + 4 <= args.N) {
            float4 *o4 = reinterpret_cast<float4 *>(o);
            if (args.epilogue == EPI_ADD) {
                float4 t = *o4;
                f[0] += t.x; f[1] += t.y; f[2] += t.z; f[3] += t.w;
            }
            *o4 = make_float4(f[0], f[1], f[2], f[3]);
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (n0 + j < args.N) {
                    if (args.epilogue == EPI_ADD) o[j] += f[j];
                    else o[j] = f[j];
                }
            }
        }
    }
}

template <int NP, int BN, int STAGES>
__global__ void __launch_bounds__(kGemmThreads, 1)
plane_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                  const GemmArgs args) {
    using C = Cfg<NP, BN, STAGES>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // SWIZZLE_128B atoms need 1024 B
    const uint32_t bar_base = smem_base + STAGES * C::STAGE_BYTES;
    // barrier map (8 B each): full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2], then the TMEM address
    const uint32_t full_bar = bar_base, empty_bar = bar_base + 8 * STAGES;
    const uint32_t tfull_bar = bar_base + 16 * STAGES, tempty_bar = tfull_bar + 16;
    const uint32_t tmem_slot = tempty_bar + 16;
    uint32_t *tmem_slot_ptr =
        (uint32_t *)(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int num_tiles = args.num_m_tiles * args.num_n_tiles;
    // The K loop is cut into chunks of k_chunk k-blocks.  Each chunk is accumulated by the tensor
    // core into one of the two TMEM stages (fresh accumulator), then drained by the epilogue warps
    // into round-to-nearest fp32 register accumulators while the next chunk runs in the other
    // stage.  Reason: tcgen05 accumulates with truncation, a bias of about -1.1e-9 per K element
    // (measured); short chunks keep it at the level of fp32 rounding.
    const int num_chunks = (args.num_k_blocks + args.k_chunk - 1) / args.k_chunk;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar + 8 * s, 1);
            mbar_init(empty_bar + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(tfull_bar + 8 * a, 1);
            mbar_init(tempty_bar + 8 * a, kNumEpiWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 1) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ================= TMA producer =================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                int m_blk, n_blk;
                tile_coords(tile, args, m_blk, n_blk);
                for (int kb = 0; kb < args.num_k_blocks; ++kb) {
                    mbar_wait(empty_bar + 8 * stage, phase ^ 1u);
                    const uint32_t fb = full_bar + 8 * stage;
                    mbar_expect_tx(fb, C::STAGE_BYTES);
                    const uint32_t sa = smem_base + stage * C::STAGE_BYTES;
#pragma unroll
                    for (int pl = 0; pl < NP; ++pl)
                        tma_load_3d(sa + pl * A_PLANE_BYTES, &tmA, fb, kb * BLOCK_K, m_blk * BLOCK_M, pl);
                    tma_load_2d(sa + NP * A_PLANE_BYTES, &tmB, fb, kb * BLOCK_K, n_blk * BN);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer =================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                for (int ch = 0; ch < num_chunks; ++ch) {
                    mbar_wait(tempty_bar + 8 * acc, acc_phase ^ 1u);     // epilogue has drained this stage
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + (uint32_t)(acc * BN);
                    const int kb_end = min(args.num_k_blocks, (ch + 1) * args.k_chunk);
                    for (int kb = ch * args.k_chunk; kb < kb_end; ++kb) {
                        mbar_wait(full_bar + 8 * stage, phase);
                        tc_fence_after();
                        const uint32_t sa = smem_base + stage * C::STAGE_BYTES;
                        const uint64_t bdesc0 = umma_desc_sw128(sa + NP * A_PLANE_BYTES);
                        const uint32_t first = (kb == ch * args.k_chunk) ? 0u : 1u;
#pragma unroll
                        for (int pl = 0; pl < NP; ++pl) {
                            const uint64_t adesc0 = umma_desc_sw128(sa + pl * A_PLANE_BYTES);
#pragma unroll
                            for (int k = 0; k < BLOCK_K / UMMA_K; ++k) {
                                // advancing 16 elements along K inside the swizzle row = +32 B = +2 in the
                                // (>>4) start-address field
                                umma_f16(d_tmem, adesc0 + (uint64_t)(2 * k), bdesc0 + (uint64_t)(2 * k), args.idesc,
                                         (pl | k) != 0 ? 1u : first);
                            }
                        }
                        umma_commit(empty_bar + 8 * stage);              // smem slot free once these MMAs retire
                        if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                    }
                    umma_commit(tfull_bar + 8 * acc);                    // this chunk's partial sums are complete
                    if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
                }
            }
        }
    } else {
        // ================= epilogue warps 2..9 =================
        // TMEM lanes 32*quarter .. +31 are the only ones this warp can read; two warps share a quarter
        // and split the BN columns between them.
        constexpr int CW = BN / 2;                       // columns per epilogue warp
        const int quarter = warp & 3;
        const int half = (warp - 2) >> 2;
        int acc = 0;
        uint32_t acc_phase = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            int m_blk, n_blk;
            tile_coords(tile, args, m_blk, n_blk);
            float racc[CW];
#pragma unroll
            for (int j = 0; j < CW; ++j) racc[j] = 0.f;
            const int m = m_blk * BLOCK_M + quarter * 32 + lane;
            for (int ch = 0; ch < num_chunks; ++ch) {
                // per-(row, chunk) power-of-two factor of the scaled fp16 planes (exact); loaded before the wait
                const float sc = (args.chunk_scale && m < args.M) ? args.chunk_scale[(size_t)ch * args.M + m] : 1.f;
                mbar_wait(tfull_bar + 8 * acc, acc_phase);
                tc_fence_after();
                const uint32_t t_addr = tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(acc * BN + half * CW);
#pragma unroll
                for (int c = 0; c < CW; c += 32) {
                    uint32_t v[32];
                    tmem_ld32(t_addr + (uint32_t)c, v);
#pragma unroll
                    for (int j = 0; j < 32; ++j) racc[c + j] = fmaf(__uint_as_float(v[j]), sc, racc[c + j]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty_bar + 8 * acc);
                if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
            }
            if (m < args.M) {
                const float rv = args.rowv ? args.rowv[m] : 0.f;
                store_row<CW>(racc, args, m, n_blk * BN + half * CW, rv);
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 512);
    }
}

// ------------------------------------------------------------------ CTA-pair version (cta_group::2)
// The one-CTA kernel above is bound by the L2 -> shared-memory feed, not by the tensor pipe: a
// 128 x 256 tile with two A planes pulls 64 KB per k-block of 1024 MMA cycles = 64 B/clk/SM, and
// the chip delivers about 6300 B/clk in all = 43 B/clk/SM (B300_MICROARCH.md "TMA chip-throughput").
// Here two CTAs of a cluster (the two SMs of a TPC) share one 256 x BN tile: each loads its own 128
// rows of the A planes and HALF of the B tile, and one tcgen05.mma.cta_group::2 (M = 256) issued by
// the leader CTA reads both halves of B, so the feed drops to 48 B/clk/SM for BN = 256.
// Same roles, same K-chunked TMEM accumulation; what changes is the synchronisation:
//   full[s]    lives in the leader; the TMA of BOTH CTAs signals it (.cta_group::2, peer bit cleared)
//   empty[s]   one per CTA, released by a multicast tcgen05.commit from the leader
//   tfull[a]   one per CTA, same multicast commit
//   tempty[a]  lives in the leader, counts the epilogue warps of both CTAs (remote arrive)
constexpr uint32_t kPeerBitMask = 0xFEFFFFFFu;      // shared::cluster address of the same offset in the even CTA

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_id_x() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t num_clusters_x() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void tma_load_2d_2sm(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar & kPeerBitMask), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_load_3d_2sm(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar & kPeerBitMask), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void umma_f16_2sm(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrives on the barrier at this offset in BOTH CTAs once every MMA issued so far has completed
__device__ __forceinline__ void umma_commit_2sm(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(bar), "h"((uint16_t)3) : "memory");
}
__device__ __forceinline__ void mbar_arrive_leader(uint32_t bar) {
    // relaxed: what is ordered is this warp's tcgen05.ld before the leader's next tcgen05.mma, and the tcgen05 fences
    // on both sides do that; a release at cluster scope compiles to a full MEMBAR.GPU, which waits for the tile's
    // result stores to drain.
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar & kPeerBitMask) : "memory");
}
__device__ __forceinline__ void tmem_alloc_2sm(uint32_t dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_2sm(uint32_t addr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}

constexpr int PAIR_M = 2 * BLOCK_M;            // rows of a pair tile
constexpr int kGroupPairM = 4;                 // rasterisation: 4 pair-rows (1024 rows) share each n sweep

constexpr int kOutTileBytes = 32 * 128;        // a warp's 32 x 32 fp32 staging tile (one SWIZZLE_128B box)
template <int NP, int BN, int STAGES, int STATS>
struct Cfg2 {
    static constexpr int HB = BN / 2;                                 // B rows held by each CTA
    static constexpr int B_BYTES = HB * BLOCK_K * 2;
    static constexpr int STAGE_BYTES = NP * A_PLANE_BYTES + B_BYTES;  // per CTA
    static constexpr int OUT_BYTES = kNumEpiWarps * kOutTileBytes;    // after the ring, 1024-byte aligned
    static constexpr int BAR_BYTES = 256;
    static constexpr int LW_BYTES = STATS ? kNumEpiWarps * 128 : 0;   // log w of a warp's 32 rows
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + OUT_BYTES + BAR_BYTES + LW_BYTES + 1024;
    static_assert(STAGE_BYTES % 1024 == 0, "the staging tiles must keep the 1024-byte swizzle alignment");
    static_assert(SMEM_BYTES <= 232448, "exceeds the 227 KB of shared memory per CTA");
    static_assert(2 * BN <= 512, "two accumulator stages must fit the 512 TMEM columns");
    static_assert(BN % 64 == 0 && BN <= 256, "UMMA N for M = 256; two epilogue warps per lane quarter");
    static_assert(HB % 8 == 0, "whole swizzle atoms");
};

__device__ __forceinline__ void tma_store_2d(const CUtensorMap *map, uint32_t src, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
                 ::"l"(map), "r"(src), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_reduce_add_2d(const CUtensorMap *map, uint32_t src, int c0, int c1) {
    asm volatile("cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3}], [%1];"
                 ::"l"(map), "r"(src), "r"(c0), "r"(c1) : "memory");
}

// Final phase of a tile in the pair kernel.  The warp holds 32 rows x CW columns, one row per lane.  Measured
// (clock64 around this phase, C2): with per-lane global stores it took 20-33 thousand cycles per tile, more than
// the two TMEM stages of MMA work that can hide it, because every L1 wavefront queues behind the tensor core's
// operand reads and the TMA fills; so the phase is built to issue as few wavefronts as possible.  Each 32 x 32
// block is written once to a 4 KB shared-memory tile in the SWIZZLE_128B pattern (8 conflict-free 16-byte stores
// per lane) and leaves as ONE asynchronous TMA store (or reduce-add for EPI_ADD), which also clips the ragged
// edges of the matrix.  The log-likelihood variant (STATS) reads the same tile back transposed (lane = column)
// for the first sweep of the normalisation: per-column max and sum of exp of a = L + log w_r over the 32 rows,
// one partial per (32-row block, column), in one online pass.  a is formed from the stored fp32 L exactly as
// normalize_kernel forms it.  Rows beyond M are staged as -inf (STATS) and never reach memory.
template <int CW, int STATS>   // STATS: 0 = store only, 1 = + column statistics of L, 2 = + those of the Gaussian Q
__device__ __forceinline__ void tile_out(const float (&racc)[CW], const GemmArgs &args, const CUtensorMap *tmC, int m,
                                         int row0, int n_base, uint8_t *tile, float *lwbuf, int lane,
                                         const typename GaussOf<STATS>::type &gp) {
    if (row0 >= args.M) return;                                     // warp-uniform: nothing of this block exists
    const bool live = m < args.M;
    const float rv = (live && args.rowv) ? args.rowv[m] : 0.f;
    // eq. (2.5) divides a whole row by s[r]: one reciprocal per row.  (A division per element ran at 280 cycles
    // each here: most numerators are subnormal and take the slow path of the IEEE division routine.)
    const float inv = rv > 0.f ? 1.f / rv : 0.f;
    const bool inv_ok = !(rv > 0.f) || inv < 3.0e38f;              // s[r] so small that 1/s overflows: divide
    const uint32_t tile_s = smem_u32(tile);
    // Gaussian model: Q = B^2 g_d + (-C_r / (2 sigma^2)), g_d = 1 / (2 sigma^2 A_d): the row term joins log w_r as the
    // row's "log weight", the element term B^2 g_d plays the role of L in the reference-pair statistics
    constexpr bool gauss = STATS == 2;
    const bool uniform = args.weight == nullptr && !gauss;
    if constexpr (STATS == 1) {
        if (!uniform) lwbuf[lane] = live ? logf(args.weight[m]) : 0.f;
    } else if constexpr (STATS == 2) {
        const float lw = args.weight ? logf(live ? args.weight[m] : 1.f) : args.log_uniform;
        lwbuf[lane] = live ? gauss_row_term(lw, rv, gp.inv2s2) : -INFINITY;
    }
    const size_t so = (size_t)(row0 >> 5) * args.ld_stat;
#pragma unroll
    for (int c = 0; c < CW; c += 32) {
        if (n_base + c >= args.N) break;                            // warp-uniform
        if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the tile is free again
        __syncwarp();
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            float f[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float v = racc[c + 4 * k + j];
                if (args.epilogue == EPI_SUB_ROW) f[j] = v - rv;
                else if (args.epilogue == EPI_DIV_ROW) f[j] = inv_ok ? v * inv : (rv > 0.f ? v / rv : 0.f);
                else f[j] = v;
                if (STATS && !live) f[j] = gauss ? 0.f : -INFINITY;
            }
            *reinterpret_cast<float4 *>(tile + lane * 128 + ((k ^ (lane & 7)) << 4)) = make_float4(f[0], f[1], f[2], f[3]);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {
            if (args.epilogue == EPI_ADD) tma_reduce_add_2d(tmC, tile_s, n_base + c, row0);
            else tma_store_2d(tmC, tile_s, n_base + c, row0);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (STATS) {
            const int col = n_base + c + lane;
            const float *colp = reinterpret_cast<const float *>(tile) + (lane & 3);
            const int chunk = lane >> 2;
            float g_col = 0.f;
            if constexpr (gauss) {
                if (col < args.N) g_col = gp.g[col];
            }
            // online statistics over the 32 rows, four rows per step, as a reference pair (mL, mw) = (L, log w) of
            // the row with the largest L + log w and z = sum exp((L - mL) + (log w - mw)): see ColStat in
            // emc_normalize.cu for why the two differences are taken separately.  Rows beyond M carry L = -inf.
            float mL = -INFINITY, mw = 0.f, z = 0.f;
            if (uniform) {
                // log w is the same for every row: it drops out of the differences, the reference is the largest L
                mw = args.log_uniform;
#pragma unroll
                for (int i0 = 0; i0 < 32; i0 += 4) {
                    float l4[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) l4[k] = colp[(i0 + k) * 32 + ((chunk ^ ((i0 + k) & 7)) << 2)];
                    // row 0 of a block exists, so mn is finite from the first step on; exp(-inf - mn) = 0
                    const float mn = fmaxf(fmaxf(mL, fmaxf(l4[0], l4[1])), fmaxf(l4[2], l4[3]));
                    z = z * __expf(mL - mn) + ((__expf(l4[0] - mn) + __expf(l4[1] - mn)) + (__expf(l4[2] - mn) + __expf(l4[3] - mn)));
                    mL = mn;
                }
            } else {
#pragma unroll 2
                for (int i0 = 0; i0 < 32; i0 += 4) {
                    float l4[4], w4[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const int i = i0 + k;
                        l4[k] = colp[i * 32 + ((chunk ^ (i & 7)) << 2)];
                        if constexpr (gauss) l4[k] = gauss_elem_term(l4[k], g_col);
                        w4[k] = lwbuf[i];
                    }
                    float bL = mL, bw = mw, bkey = mL + mw;
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const float key = l4[k] + w4[k];
                        if (key > bkey) { bkey = key; bL = l4[k]; bw = w4[k]; }
                    }
                    if (bL == -INFINITY) continue;                      // nothing but -inf so far (zero weights)
                    float add = 0.f;
#pragma unroll
                    for (int k = 0; k < 4; ++k) add += __expf((l4[k] - bL) + (w4[k] - bw));
                    z = z * __expf((mL - bL) + (mw - bw)) + add;
                    mL = bL;
                    mw = bw;
                }
            }
            if (col < args.N) {
                args.stat_m[so + col] = mL;
                args.stat_w[so + col] = mw;
                args.stat_z[so + col] = z;
            }
        }
    }
}

__device__ __forceinline__ void pair_tile_coords(int tile, const GemmArgs &a, int &m_blk, int &n_blk) {
    const int per_group = kGroupPairM * a.num_n_tiles;
    const int group = tile / per_group;
    const int first_m = group * kGroupPairM;
    const int gm = min(a.num_m_tiles - first_m, kGroupPairM);
    const int t = tile - group * per_group;
    m_blk = first_m + t % gm;
    n_blk = t / gm;
}

// args.num_m_tiles counts PAIR tiles (256 rows)
template <int NP, int BN, int STAGES, int STATS>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kGemmThreads, 1)
plane_gemm_pair_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                       const __grid_constant__ CUtensorMap tmC, const GemmArgs args,
                       const typename GaussOf<STATS>::type gp) {
    using C = Cfg2<NP, BN, STAGES, STATS>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t out_base = smem_base + STAGES * C::STAGE_BYTES;            // 8 staging tiles of 4 KB
    const uint32_t bar_base = out_base + C::OUT_BYTES;
    const uint32_t full_bar = bar_base, empty_bar = bar_base + 8 * STAGES;
    const uint32_t tfull_bar = bar_base + 16 * STAGES, tempty_bar = tfull_bar + 16;
    const uint32_t tmem_slot = tempty_bar + 16;
    uint32_t *tmem_slot_ptr = (uint32_t *)(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const bool leader = rank == 0;
    const int num_tiles = args.num_m_tiles * args.num_n_tiles;
    const int first_tile = (int)cluster_id_x(), tile_step = (int)num_clusters_x();
    const int num_chunks = (args.num_k_blocks + args.k_chunk - 1) / args.k_chunk;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmC) : "memory");
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar + 8 * s, 1);
            mbar_init(empty_bar + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(tfull_bar + 8 * a, 1);
            mbar_init(tempty_bar + 8 * a, 2 * kNumEpiWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 1) tmem_alloc_2sm(tmem_slot, 512);
    tc_fence_before();
    cluster_sync_all();                           // both CTAs' barriers exist before anyone signals them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ================= TMA producer (both CTAs) =================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = first_tile; tile < num_tiles; tile += tile_step) {
                int m_blk, n_blk;
                pair_tile_coords(tile, args, m_blk, n_blk);
                const int m0 = m_blk * PAIR_M + (int)rank * BLOCK_M;
                const int n0 = n_blk * BN + (int)rank * C::HB;
                for (int kb = 0; kb < args.num_k_blocks; ++kb) {
                    mbar_wait(empty_bar + 8 * stage, phase ^ 1u);
                    const uint32_t fb = full_bar + 8 * stage;
                    if (leader) mbar_expect_tx(fb, 2 * C::STAGE_BYTES);   // the bytes of both CTAs
                    const uint32_t sa = smem_base + stage * C::STAGE_BYTES;
#pragma unroll
                    for (int pl = 0; pl < NP; ++pl)
                        tma_load_3d_2sm(sa + pl * A_PLANE_BYTES, &tmA, fb, kb * BLOCK_K, m0, pl);
                    tma_load_2d_2sm(sa + NP * A_PLANE_BYTES, &tmB, fb, kb * BLOCK_K, n0);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer (leader CTA only) =================
        if (leader && lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (int tile = first_tile; tile < num_tiles; tile += tile_step) {
                for (int ch = 0; ch < num_chunks; ++ch) {
                    mbar_wait(tempty_bar + 8 * acc, acc_phase ^ 1u);     // both epilogues have drained this stage
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + (uint32_t)(acc * BN);
                    const int kb_end = min(args.num_k_blocks, (ch + 1) * args.k_chunk);
                    for (int kb = ch * args.k_chunk; kb < kb_end; ++kb) {
                        mbar_wait(full_bar + 8 * stage, phase);
                        tc_fence_after();
                        const uint32_t sa = smem_base + stage * C::STAGE_BYTES;
                        const uint64_t bdesc0 = umma_desc_sw128(sa + NP * A_PLANE_BYTES);
                        const uint32_t first = (kb == ch * args.k_chunk) ? 0u : 1u;
#pragma unroll
                        for (int pl = 0; pl < NP; ++pl) {
                            const uint64_t adesc0 = umma_desc_sw128(sa + pl * A_PLANE_BYTES);
#pragma unroll
                            for (int k = 0; k < BLOCK_K / UMMA_K; ++k)
                                umma_f16_2sm(d_tmem, adesc0 + (uint64_t)(2 * k), bdesc0 + (uint64_t)(2 * k), args.idesc,
                                             (pl | k) != 0 ? 1u : first);
                        }
                        umma_commit_2sm(empty_bar + 8 * stage);          // frees the slot in both CTAs
                        if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                    }
                    umma_commit_2sm(tfull_bar + 8 * acc);                // partial sums complete in both CTAs
                    if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
                }
            }
        }
    } else {
        // ================= epilogue warps 2..9 (both CTAs; each drains its own 128 rows) =================
        constexpr int CW = BN / 2;
        const int quarter = warp & 3;
        const int half = (warp - 2) >> 2;
        int acc = 0;
        uint32_t acc_phase = 0;
        for (int tile = first_tile; tile < num_tiles; tile += tile_step) {
            int m_blk, n_blk;
            pair_tile_coords(tile, args, m_blk, n_blk);
            float racc[CW];
#pragma unroll
            for (int j = 0; j < CW; ++j) racc[j] = 0.f;
            const int m = m_blk * PAIR_M + (int)rank * BLOCK_M + quarter * 32 + lane;
            for (int ch = 0; ch < num_chunks; ++ch) {
                const float sc = (args.chunk_scale && m < args.M) ? args.chunk_scale[(size_t)ch * args.M + m] : 1.f;
                mbar_wait(tfull_bar + 8 * acc, acc_phase);
                tc_fence_after();
                const uint32_t t_addr = tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(acc * BN + half * CW);
#pragma unroll
                for (int c = 0; c < CW; c += 32) {
                    uint32_t v[32];
                    tmem_ld32(t_addr + (uint32_t)c, v);
#pragma unroll
                    for (int j = 0; j < 32; ++j) racc[c + j] = fmaf(__uint_as_float(v[j]), sc, racc[c + j]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_leader(tempty_bar + 8 * acc);
                if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
            }
            if (args.tma_out) {
                uint8_t *tile = smem_raw + (out_base - smem_u32(smem_raw)) + (warp - 2) * kOutTileBytes;
                float *lwbuf = reinterpret_cast<float *>(smem_raw + (bar_base + C::BAR_BYTES - smem_u32(smem_raw))) +
                               (warp - 2) * 32;
                tile_out<CW, STATS>(racc, args, &tmC, m, m_blk * PAIR_M + (int)rank * BLOCK_M + quarter * 32,
                                    n_blk * BN + half * CW, tile, lwbuf, lane, gp);
            } else if (m < args.M) {               // misaligned output: per-lane stores
                const float rv = args.rowv ? args.rowv[m] : 0.f;
                store_row<CW>(racc, args, m, n_blk * BN + half * CW, rv);
            }
        }
        if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // staging tiles read, results written
    }

    tc_fence_before();
    cluster_sync_all();                           // the peer may still be reading operands / signalling barriers here
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc_2sm(tmem_base, 512);
    }
}

// ------------------------------------------------------------------ plain CUDA-core version (EMC_DEBUG_SIMT)
__device__ __forceinline__ float load16(const void *p, size_t i, int fmt) {
    const uint16_t u = ((const uint16_t *)p)[i];
    return fmt == FMT_F16 ? __half2float(__ushort_as_half(u)) : __uint_as_float((uint32_t)u << 16);
}

__global__ void simt_plane_gemm_kernel(GemmProblem g) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = blockIdx.y;
    if (n >= g.N || m >= g.M) return;
    float acc = 0.f;
    const int chunk = kChunkKBlocks * BLOCK_K;
    for (int k0 = 0; k0 < g.K; k0 += chunk) {
        float part = 0.f;
        for (int pl = 0; pl < g.n_planes; ++pl)
            for (int k = k0; k < min(g.K, k0 + chunk); ++k)
                part += load16(g.A, pl * g.plane_stride + (size_t)m * g.lda + k, g.a_fmt) *
                        load16(g.B, (size_t)n * g.ldb + k, g.b_fmt);
        acc += part * (g.chunk_scale ? g.chunk_scale[(size_t)(k0 / chunk) * g.M + m] : 1.f);
    }
    float *o = g.out + (size_t)m * g.ld_out + n;
    const float rv = g.rowv ? g.rowv[m] : 0.f;
    switch (g.epilogue) {
        case EPI_SUB_ROW: *o = acc - rv; break;
        case EPI_STORE: *o = acc; break;
        case EPI_ADD: *o += acc; break;
        default: *o = rv > 0.f ? acc / rv : 0.f; break;
    }
}

// ------------------------------------------------------------------ host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

emc_status get_encode_fn(EncodeTiledFn *out) {
    static EncodeTiledFn cached = nullptr;
    if (!cached) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        EMC_TRY_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (qres != cudaDriverEntryPointSuccess || !fn) return cuda_fail(cudaErrorUnknown, "cuTensorMapEncodeTiled entry point");
        cached = (EncodeTiledFn)fn;
    }
    *out = cached;
    return EMC_OK;
}

emc_status make_map(CUtensorMap *map, const void *base, PlaneFormat fmt, int rank, const cuuint64_t *dims,
                    const cuuint64_t *strides_bytes, const cuuint32_t *box) {
    EncodeTiledFn enc;
    EMC_TRY(get_encode_fn(&enc));
    const cuuint32_t ones[3] = {1, 1, 1};
    CUresult r = enc(map, fmt == FMT_F16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16,
                     (cuuint32_t)rank, const_cast<void *>(base), dims, strides_bytes, box, ones,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cuda_fail(cudaErrorInvalidValue, "cuTensorMapEncodeTiled");
    return EMC_OK;
}

// fp32 output [rows][ld] as 32 x 32 boxes in the SWIZZLE_128B pattern (tile_out)
emc_status make_out_map(CUtensorMap *map, const float *base, int rows, int cols, int ld) {
    EncodeTiledFn enc;
    EMC_TRY(get_encode_fn(&enc));
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
    const cuuint32_t box[2] = {32, 32};
    const cuuint32_t ones[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(base), dims, strides, box, ones,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cuda_fail(cudaErrorInvalidValue, "cuTensorMapEncodeTiled (output)");
    return EMC_OK;
}

int num_sms() {
    static int sms = 0;
    if (!sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (sms <= 0) sms = 148;
    }
    return sms;
}

template <int NP, int BN, int STAGES>
emc_status launch_tc(const GemmProblem &g, cudaStream_t st) {
    using C = Cfg<NP, BN, STAGES>;
    CUtensorMap tmA, tmB;
    {
        const cuuint64_t dims[3] = {(cuuint64_t)g.K, (cuuint64_t)g.M, (cuuint64_t)NP};
        const cuuint64_t strides[2] = {(cuuint64_t)g.lda * 2, (cuuint64_t)g.plane_stride * 2};
        const cuuint32_t box[3] = {BLOCK_K, BLOCK_M, 1};
        EMC_TRY(make_map(&tmA, g.A, g.a_fmt, 3, dims, strides, box));
    }
    {
        const cuuint64_t dims[2] = {(cuuint64_t)g.K, (cuuint64_t)g.N};
        const cuuint64_t strides[1] = {(cuuint64_t)g.ldb * 2};
        const cuuint32_t box[2] = {BLOCK_K, BN};
        EMC_TRY(make_map(&tmB, g.B, g.b_fmt, 2, dims, strides, box));
    }
    GemmArgs a;
    a.M = g.M; a.N = g.N; a.K = g.K;
    a.num_m_tiles = ceil_div(g.M, BLOCK_M);
    a.num_n_tiles = ceil_div(g.N, BN);
    a.num_k_blocks = ceil_div(g.K, BLOCK_K);
    a.out = g.out; a.ld_out = g.ld_out; a.rowv = g.rowv; a.epilogue = g.epilogue;
    a.k_chunk = g.k_chunk > 0 ? g.k_chunk : kChunkKBlocks;
    a.chunk_scale = g.chunk_scale;
    a.vec_ok = (g.ld_out % 4 == 0) && (((uintptr_t)g.out & 15) == 0);
    a.stat_m = a.stat_w = a.stat_z = nullptr; a.ld_stat = 0; a.weight = nullptr; a.log_uniform = 0.f; a.tma_out = 0;
    // instruction descriptor (kind::f16): D = F32 [4,6); A format [7,10); B format [10,13); both K-major;
    // N >> 3 in [17,23); M >> 4 in [24,29)
    a.idesc = (1u << 4) | ((uint32_t)g.a_fmt << 7) | ((uint32_t)g.b_fmt << 10) | ((uint32_t)(BN >> 3) << 17) |
              ((uint32_t)(BLOCK_M >> 4) << 24);
    auto kern = plane_gemm_kernel<NP, BN, STAGES>;
    static bool attr_set = false;
    if (!attr_set) {
        EMC_TRY_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
        attr_set = true;
    }
    const int tiles = a.num_m_tiles * a.num_n_tiles;
    const int grid = tiles < num_sms() ? tiles : num_sms();
    kern<<<grid, kGemmThreads, C::SMEM_BYTES, st>>>(tmA, tmB, a);
    EMC_LAUNCHED();
    return EMC_OK;
}

int max_pair_clusters(const void *kern, int smem_bytes) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * 74);
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = (size_t)smem_bytes;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n <= 0) {
        cudaGetLastError();
        n = num_sms() / 2;
    }
    return n;
}

template <int NP, int BN, int STAGES, int STATS>
emc_status launch_tc_pair(const GemmProblem &g, cudaStream_t st) {
    using C = Cfg2<NP, BN, STAGES, STATS>;
    CUtensorMap tmA, tmB;
    {
        const cuuint64_t dims[3] = {(cuuint64_t)g.K, (cuuint64_t)g.M, (cuuint64_t)NP};
        const cuuint64_t strides[2] = {(cuuint64_t)g.lda * 2, (cuuint64_t)g.plane_stride * 2};
        const cuuint32_t box[3] = {BLOCK_K, BLOCK_M, 1};
        EMC_TRY(make_map(&tmA, g.A, g.a_fmt, 3, dims, strides, box));
    }
    {
        const cuuint64_t dims[2] = {(cuuint64_t)g.K, (cuuint64_t)g.N};
        const cuuint64_t strides[1] = {(cuuint64_t)g.ldb * 2};
        const cuuint32_t box[2] = {BLOCK_K, C::HB};
        EMC_TRY(make_map(&tmB, g.B, g.b_fmt, 2, dims, strides, box));
    }
    GemmArgs a;
    a.M = g.M; a.N = g.N; a.K = g.K;
    a.num_m_tiles = ceil_div(g.M, PAIR_M);
    a.num_n_tiles = ceil_div(g.N, BN);
    a.num_k_blocks = ceil_div(g.K, BLOCK_K);
    a.out = g.out; a.ld_out = g.ld_out; a.rowv = g.rowv; a.epilogue = g.epilogue;
    a.k_chunk = g.k_chunk > 0 ? g.k_chunk : kChunkKBlocks;
    a.chunk_scale = g.chunk_scale;
    a.vec_ok = (g.ld_out % 4 == 0) && (((uintptr_t)g.out & 15) == 0);
    a.idesc = (1u << 4) | ((uint32_t)g.a_fmt << 7) | ((uint32_t)g.b_fmt << 10) | ((uint32_t)(BN >> 3) << 17) |
              ((uint32_t)(PAIR_M >> 4) << 24);
    a.stat_m = g.stat_m; a.stat_w = g.stat_w; a.stat_z = g.stat_z; a.ld_stat = g.ld_stat; a.weight = g.weight;
    a.log_uniform = g.log_uniform;
    a.tma_out = a.vec_ok;
    if (STATS && !a.tma_out) return EMC_ERR_ARG;             // gemm_fuses_stats() said no
    CUtensorMap tmC = tmA;                                    // placeholder when the output is not TMA-addressable
    if (a.tma_out) EMC_TRY(make_out_map(&tmC, g.out, g.M, g.N, g.ld_out));
    auto kern = plane_gemm_pair_kernel<NP, BN, STAGES, STATS>;
    static int clusters = 0;
    if (!clusters) {
        EMC_TRY_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
        clusters = max_pair_clusters((const void *)kern, C::SMEM_BYTES);
    }
    const int tiles = a.num_m_tiles * a.num_n_tiles;
    const int grid = 2 * (tiles < clusters ? tiles : clusters);
    typename GaussOf<STATS>::type gp;
    if constexpr (STATS == 2) { gp.g = g.gauss_g; gp.inv2s2 = g.inv2s2; }
    kern<<<grid, kGemmThreads, C::SMEM_BYTES, st>>>(tmA, tmB, tmC, a, gp);     // cluster size is a kernel attribute
    EMC_LAUNCHED();
    return EMC_OK;
}

}  // namespace

bool gemm_fuses_stats(const GemmProblem &g, bool simt_debug) {
    const bool aligned = (g.ld_out % 4 == 0) && (((uintptr_t)g.out & 15) == 0);      // the output goes out by TMA
    return g.stat_m && g.stat_w && g.stat_z && g.rowv && (g.epilogue == EPI_SUB_ROW || g.epilogue == EPI_GAUSS) && g.n_planes == 2 && !g.one_cta && !simt_debug &&
           aligned;
}

emc_status launch_plane_gemm(const GemmProblem &g, bool simt_debug, cudaStream_t st) {
    if (g.M <= 0 || g.N <= 0 || g.K <= 0) return EMC_ERR_ARG;
    if (g.lda % 8 || g.ldb % 8 || g.plane_stride % 8 || ((uintptr_t)g.A & 15) || ((uintptr_t)g.B & 15)) return EMC_ERR_ARG;
    if (simt_debug) {
        dim3 grid(ceil_div(g.N, 128), g.M);
        simt_plane_gemm_kernel<<<grid, 128, 0, st>>>(g);
        EMC_LAUNCHED();
        return EMC_OK;
    }
    if (g.epilogue == EPI_GAUSS && !(g.stat_m && g.gauss_g && g.n_planes == 2 && !g.one_cta && !simt_debug))
        return EMC_ERR_UNSUPPORTED;                              // the Gaussian statistics exist in the pair kernel only
    if (g.n_planes == 2 && !g.one_cta) {
        // CTA pairs; tile width by wave quantisation: time ~ waves(BN) x BN (one pair per TPC, tiles of equal cost)
        const int mt = ceil_div(g.M, PAIR_M), pairs = num_sms() / 2;
        const long c256 = (long)ceil_div(mt * ceil_div(g.N, 256), pairs) * 256;
        const long c192 = (long)ceil_div(mt * ceil_div(g.N, 192), pairs) * 192;
        if (g.stat_m && g.epilogue == EPI_GAUSS)
            return c192 < c256 ? launch_tc_pair<2, 192, 4, 2>(g, st) : launch_tc_pair<2, 256, 4, 2>(g, st);
        if (g.stat_m)
            return c192 < c256 ? launch_tc_pair<2, 192, 4, 1>(g, st) : launch_tc_pair<2, 256, 4, 1>(g, st);
        return c192 < c256 ? launch_tc_pair<2, 192, 4, 0>(g, st) : launch_tc_pair<2, 256, 4, 0>(g, st);
    }
    if (g.n_planes == 2) {
        // tile width by wave quantisation: time ~ waves(BN) x BN (one CTA per SM, tiles of equal cost)
        const int mt = ceil_div(g.M, BLOCK_M), sms = num_sms();
        const long c256 = (long)ceil_div(mt * ceil_div(g.N, 256), sms) * 256;
        const long c192 = (long)ceil_div(mt * ceil_div(g.N, 192), sms) * 192;
        return c192 < c256 ? launch_tc<2, 192, 4>(g, st) : launch_tc<2, 256, 3>(g, st);
    }
    return EMC_ERR_UNSUPPORTED;
}

}  // namespace emc
