// a4: grouped SwiGLU expert FFN over cache slots -- tcgen05 / TMEM / TMA kernel for sm_100a.
//
// ONE launch per wave: a persistent, warp-specialised grouped GEMM that runs BOTH GEMMs of the wave's experts.  Its work
// list holds the GEMM1 units (x -> h) followed by the GEMM2 units (h -> y); a GEMM2 unit waits -- in its TMA producer
// only, after the weight box of its first stage is already on its way -- until the GEMM1 units of its own token tile have
// stored their h columns (one release counter per token tile, bumped once per weight tile).  There is no launch boundary,
// no ramp and no tail between the two GEMMs: GEMM2 of the experts that finished early overlaps GEMM1 of the rest, h
// is read back out of L2, and a decode wave streams W13 and Wd as one uninterrupted pass over the expert.
// Both GEMMs are computed TRANSPOSED ("swap-AB"): the weight rows are the MMA M side (always full 128-lane
// accumulators), the ragged token rows are the MMA N side, whose granularity is 16 -- so an expert with M_e routed rows
// costs ceil16(M_e) MMA columns, not a multiple of 128 rows (BASELINE.json cfg 2: 4096 routed rows occupy 4144 MMA columns
// instead of 4608 rows).
//   D[w, t] = sum_k W_slot(g)[w, k] . A[t, k]          (bf16 x bf16 -> fp32 in TMEM; lanes = weight rows, columns = tokens)
//   GEMM1: A = x_perm, W = packed W13 (gate/up interleaved by 128 rows): accumulator 0 = 128 gate rows, accumulator 1 =
//          the matching 128 up rows, same lanes -> epilogue h = silu(g) * u -> bf16
//   GEMM2: A = h,      W = Wd: accumulators 0 / 1 = output features [256 n, +128) / [256 n + 128, +128) -> bf16 y
// (PAPER.md L46 leaves e_i opaque; SwiGLU is BASELINE.json's choice, R4.)
//
// CTA pairs (cta_group::2): the two CTAs of a cluster work on the same token tile and on two adjacent 256-row weight
// tiles.  Each CTA loads its own weight tile (M side, 128 + 128 rows for its two accumulators) and HALF of the token
// tile (N side); one tcgen05.mma.cta_group::2 (M256 N<=256 K16) per accumulator, issued by the leader CTA, reads both
// halves, so the token operand is fetched from L2 and staged in shared memory once per pair.  Per k-step (K = 64) a
// CTA therefore pulls 32 KB of weights + <= 16 KB of tokens for 2 * n/2 * 4 tensor cycles -- 48 B/cycle at n = 256
// against 64 for a single-CTA 256 x 256 tile -- and a stage is 48 KB, which buys a 4th pipeline stage.
// Tokens past the end of the group are loaded and multiplied (their columns are never stored), token rows past the
// tensor are zero-filled by TMA.  The weight operand of a stage is ONE contiguous 32 KB box: the packed expert layout
// is tiled in streaming order (ef_internal.h), and the whole slot arena is one 2-D tensor map of 128-byte rowlets.
//
// Warp roles (384 threads, 1 CTA/SM, persistent; both CTAs unless stated):
//   warp 0     TMA producer + tile scheduler : the LEADER claims the next unit with one atomicAdd on a per-launch
//                                counter and hands it to both CTAs' roles through 4-deep smem rings (the peer's copy
//                                by one st.async that also completes its barrier); each CTA's producer then issues its own boxes,
//                                all completing on the leader's "full" barrier
//   warp 1     MMA issuer (leader only) : one lane issues the two MMAs per k-step; tcgen05.commit multicasts the
//                                "stage free" / "accumulator ready" arrivals to both CTAs
//   warp 2     TMEM allocator    : 512 columns per CTA.  A tile with > 128 tokens takes all of them (accumulators at
//                                columns 0 and 256); tiles with <= 128 tokens alternate between the two 256-column
//                                halves (accumulators at +0 and +128), so their epilogue overlaps the next tile's MMAs
//   warp 3     prologue          : token tiling of the wave's groups into shared memory
//   warps 4-11 epilogue          : tcgen05.ld 16x256b (the MMA C-fragment layout) -> SwiGLU / cast -> stmatrix.trans
//                                into a [32 tokens][128 features] staging tile -> 16-byte global stores, 256
//                                contiguous bytes per token row; warps w and w+4 share a TMEM lane quarter and
//                                take alternate 32-token chunks; "accumulator free" arrives on the leader's barrier
// Hand-backs across the pair (ring slots, drained TMEM halves) are RELAXED remote arrives: a cluster-scope release is a
// MEMBAR.GPU on this device and made the MMA lane wait ~1 us for TMEM on every unit ("hand-overs").
// Per-expert tile scheduling over ragged token counts: inside a phase units are numbered longest-first -- every
// > 128-token tile of every group (n-major inside a group, so the token tiles that share a weight tile are claimed back
// to back and hit L2) with the <= 128-token tail tiles spread among them -- and claimed dynamically (greedy list
// scheduling).
// Tail split-K: with T units on G pairs the last T mod G units of a phase (all of them when T < G -- decode,
// single-expert miss waves) would leave most SMs idle for a whole tile time, so the host splits each of those units s
// ways along K.  A split unit writes its raw fp32 accumulators to a workspace slot, then bumps the tile's arrival
// counter; the unit that arrives last sums the s partials in split order (deterministic) and runs the normal epilogue.
// No CTA ever waits for another cluster on this path; the only cross-CTA wait is a GEMM2 producer's wait for h rows,
// whose GEMM1 units were all claimed -- by CTAs that never wait themselves -- before any GEMM2 ticket was handed out.
#include <cuda_bf16.h>

#include "ef_internal.h"

namespace {

constexpr int BK = 64;                 // K elements per stage (128 bytes of bf16)
constexpr int BW = 256;                // weight rows per tile (two 128-lane accumulators)
constexpr int ACC_M = 128;             // weight rows per accumulator
constexpr int BT = 256;                // max tokens per tile
constexpr int XBOX = 64;               // token rows per TMA box
constexpr int kStages = 4;
constexpr int W_BYTES = BW * BK * 2;              // 32 KB
constexpr int XBOX_BYTES = XBOX * BK * 2;         // 8 KB
constexpr int STAGE_BYTES = W_BYTES + (BT / 2) * BK * 2;   // 48 KB: own weight tile + own half of the token tile
constexpr int kThreads = 384;
constexpr int kEpiWarps = 8;
constexpr int kSched = 4;               // depth of the tile-broadcast ring
constexpr int kTmemCols = 512;
constexpr int kSlotFloats = 2 * 128 * 256;   // LARGEST split-K workspace slot: two 128-lane x 256-column fp32 accumulators; a wave whose
                                             // token tiles are narrower uses proportionally smaller slots (PhaseArgs::ws_acc_f4)
// Epilogue staging (transpose): per column-parity group of 4 warps one [32 tokens][128 features] bf16 tile, rows
// padded by 16 B so that stmatrix rows (stride 272 B) and 16-byte read-backs are bank-conflict free
constexpr int STG_LD = ACC_M * 2 + 16;
constexpr int STG_BYTES = 32 * STG_LD;

// -DEF_KPROF: the MMA-issuing lane of every CTA accumulates the cycles it spends waiting for a tile ticket, for the
// epilogue to free TMEM and for TMA to fill a stage, and dumps them per CTA (ef_diag_kprof, diag library).  Off in normal builds.
// -DEF_KTIME (with -DEF_KPROF): instead of the wait cycles, the same five words hold a TIMELINE of the pair in globaltimer
// nanoseconds: {prologue done, first stage full, last GEMM1 unit issued, first GEMM2 stage full, last unit issued}.
#ifdef EF_KTIME
#define KTIME(...) __VA_ARGS__
#else
#define KTIME(...)
#endif
#ifdef EF_KPROF
#define KPROF(...) __VA_ARGS__
#else
#define KPROF(...)
#endif

struct __align__(8) SmemCtl {
    uint64_t full[kStages];
    uint64_t empty[kStages];
    uint64_t tmem_full[2];
    uint64_t tmem_empty[2];
    uint64_t sched_full[kSched];
    uint64_t sched_empty[kSched];
    int32_t sched_tile[kSched];
    uint32_t tmem_base;
    int32_t split_last;                   // epilogue broadcast: this unit arrived last at its split tile
    // token tiling of the wave (prologue; the same for both GEMMs): exclusive prefix sums, over the groups, of the number
    // of > 128-token ("long") tiles and of <= 128-token ("short") tail tiles; a phase multiplies them by its n_pairs_n
    int32_t tl[EF_MAX_GROUPS + 1];
    int32_t tsh[EF_MAX_GROUPS + 1];
    int16_t g_tile_rows[EF_MAX_GROUPS];   // rows per token tile of each group ...
    int16_t g_long[EF_MAX_GROUPS];        // ... and its number of long tiles
};

constexpr size_t kSmemBytes = 1024 /*align slack*/ + (size_t)kStages * STAGE_BYTES + 2 * STG_BYTES + sizeof(SmemCtl);

// ---- PTX wrappers ----------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// cluster-scope acquire: the data published before the arrive may come from the peer CTA
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of `p` (a pointer into this CTA's shared memory) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(const void* p, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(p)), "r"(rank));
    return r;
}
// Remote arrive that publishes nothing through memory (a consumer handing a ring slot or a TMEM half back: what it read is
// ordered before the arrive by its own data dependence / tcgen05.fence::before_thread_sync).  No cluster-scope release:
// that is a MEMBAR.GPU, ~1 us during which the arriving warp also waits for every global store it has in flight -- on the
// TMEM hand-over that delay is the MMA lane's.
__device__ __forceinline__ void mbar_arrive_remote_relaxed(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// ... handing back a ring slot: `read` is the value read out of the slot, an operand of the instruction only so that the
// arrive cannot issue before that shared-memory load has delivered it (the data dependence the comment above relies on)
__device__ __forceinline__ void mbar_arrive_remote_relaxed_after(uint32_t cluster_addr, int read) {
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];  // after %1" ::"r"(cluster_addr), "r"(read) : "memory");
}
// 4 bytes into the peer's shared memory that complete 4 bytes of the transaction count of a barrier there: data and
// signal in one asynchronous operation, no fence in the sender (the receiver arms the barrier with expect_tx itself)
__device__ __forceinline__ void st_async_u32(uint32_t cluster_addr, uint32_t v, uint32_t cluster_bar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.u32 [%0], %1, [%2];" ::"r"(cluster_addr), "r"(v), "r"(cluster_bar)
                 : "memory");
}
__device__ __forceinline__ void cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// TMA loads into this CTA's shared memory whose bytes complete on the LEADER's mbarrier (cluster address `bar`)
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.cta_group::2 [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(tm), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
// one lane of a converged warp
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// arrives, once the MMAs issued so far have completed, on the barrier at this offset in BOTH CTAs of the pair
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(smem_u32(bar)), "h"((uint16_t)3) : "memory");
}
// D[tmem, both CTAs] (+)= A[smem, 128 rows per CTA] . B[smem, n/2 rows per CTA]^T, M256 N(idesc) K16, bf16 -> fp32
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accum) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accum) : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, 128-byte swizzle: 8-row groups 1024 B apart (SBO), LBO unused (=1), descriptor version 1
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// kind::f16 instruction descriptor: D fp32, A/B bf16, both K-major, M = 256 (128 per CTA), N = n (multiple of 16)
__device__ __forceinline__ uint32_t make_idesc(int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)((2 * ACC_M) >> 4) << 24);
}

__device__ __forceinline__ uint16_t bf16_bits(float v) {
    __nv_bfloat16 b = __float2bfloat16_rn(v);
    return *reinterpret_cast<uint16_t*>(&b);
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}
// silu(g) * u with one MUFU op: g * sigmoid(g) = 0.5 g (1 + tanh(g / 2)); tanh.approx has ~2^-11 relative error,
// a quarter of the bf16 rounding that follows
__device__ __forceinline__ float silu_mul(float g, float u) {
    float th;
    asm("tanh.approx.f32 %0, %1;" : "=f"(th) : "f"(0.5f * g));
    const float hg = 0.5f * g;
    return fmaf(hg, th, hg) * u;
}
// 16 TMEM lanes x 32 columns: thread T gets lane T/4 (regs 4j, 4j+1) and lane T/4 + 8 (regs 4j+2, 4j+3), columns
// 8j + 2(T%4) + {0, 1} -- the MMA C-fragment layout, which is what stmatrix consumes
__device__ __forceinline__ void tc_ld16x256b_x4(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.16x256b.x4.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
}
// four 8x8 bf16 blocks, transposed on the way: smem row (16 B at the address thread 8i + r supplies for block i,
// row r) = one token, its 8 entries = the 8 TMEM lanes (features) of the block
__device__ __forceinline__ void stmatrix_x4_trans(uint32_t saddr, uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3) {
    asm volatile("stmatrix.sync.aligned.m8n8.x4.trans.shared.b16 [%0], {%1, %2, %3, %4};" ::"r"(saddr), "r"(r0), "r"(r1), "r"(r2), "r"(r3)
                 : "memory");
}
__device__ __forceinline__ void named_bar(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// The 4 warps of one column-parity group write the staged [32 tokens][128 features] tile to C with 16-byte stores
// (a half-warp covers the 256 contiguous bytes of one token row).  Barriers: staging complete / staging free again.
__device__ __forceinline__ void stage_to_global(const uint8_t* stg, uint16_t* __restrict__ C, int ldc, int64_t row0, int n_rows,
                                                int col0, int n_cols, int tid128, int bar_id) {
    named_bar(bar_id, 128);
    const int ch = tid128 & 15;
    if (col0 + ch * 8 < n_cols) {
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const int row = p * 8 + (tid128 >> 4);
            if (row < n_rows) {
                const uint4 v = *reinterpret_cast<const uint4*>(stg + row * STG_LD + ch * 16);
                *reinterpret_cast<uint4*>(C + (row0 + row) * ldc + col0 + ch * 8) = v;
            }
        }
    }
    named_bar(bar_id, 128);
}

// split-K workspace slot layout: [accumulator][column / 4][lane][4 floats] -- a warp's float4 accesses are contiguous;
// acc_f4 = float4 words per accumulator = 8 * 128 * (32-token chunks of the wave's widest tile)
__device__ __forceinline__ void ws_store32(float* slot, int acc_f4, int acc, int c, int lane128, const uint32_t (&v)[32]) {
    float4* p = reinterpret_cast<float4*>(slot) + (size_t)acc * acc_f4 + (size_t)(c * 8) * ACC_M + lane128;
#pragma unroll
    for (int i = 0; i < 8; ++i)
        p[(size_t)i * ACC_M] = make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]), __uint_as_float(v[4 * i + 2]),
                                           __uint_as_float(v[4 * i + 3]));
}
// sum over the s partial slots of a tile, in slot order; L2-only loads (the partials were written by other SMs)
__device__ __forceinline__ void ws_sum32(const float* tile_slots, int acc_f4, int s, int acc, int c, int lane128, uint32_t (&out)[32]) {
    float4 sum[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) sum[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    const float4* p = reinterpret_cast<const float4*>(tile_slots) + (size_t)acc * acc_f4 + (size_t)(c * 8) * ACC_M + lane128;
    for (int j = 0; j < s; ++j) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float4 v = __ldcg(p + (size_t)i * ACC_M);
            sum[i].x += v.x; sum[i].y += v.y; sum[i].z += v.z; sum[i].w += v.w;
        }
        p += 2 * (2 * acc_f4);           // slots alternate between the two CTAs of the pair
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        out[4 * i] = __float_as_uint(sum[i].x); out[4 * i + 1] = __float_as_uint(sum[i].y);
        out[4 * i + 2] = __float_as_uint(sum[i].z); out[4 * i + 3] = __float_as_uint(sum[i].w);
    }
}
// barrier among the 8 epilogue warps only
__device__ __forceinline__ void epi_bar() { asm volatile("bar.sync 1, 256;" ::: "memory"); }

// ---- one launch = one WAVE: both GEMMs of a set of experts --------------------------------------------------------------
// Phase 0 ("GEMM1"): A = x rows, W = packed W13 / W1, epilogue SwiGLU / ReLU, C = h workspace.
// Phase 1 ("GEMM2"): A = h rows, W = Wd,              epilogue plain,          C = y rows.
// Tickets [0, p0.total) are phase-0 units, [p0.total, p0.total + p1.total) phase-1 units; either total may be 0 (a
// single-GEMM launch: chunked expert copies gate the two GEMMs of a wave on different events, and the stage tests).
struct PhaseArgs {
    uint16_t* C;                   // output rows
    int32_t ldc, n_cols;           // leading dimension and valid columns of C
    int32_t KB;                    // k-blocks of 64
    int32_t n_tiles_n, n_pairs_n;  // 256-row weight tiles of the matrix, CTA pairs per token tile (ceil(n_tiles_n / 2))
    int32_t w_rows, base_rowlet;   // rows of the weight matrix, its first rowlet inside an arena slot
    int32_t total;                 // tickets of this phase
    int32_t n_plain, s;            // tickets [0, n_plain) are whole tiles; the rest are (tile, K part) pairs, part fastest;
                                   // s = K parts per split tile (>= 2 when any tile is split)
    int32_t ws_acc_f4;             // float4 words per accumulator in a workspace slot (a slot = 2 accumulators)
    float* ws;                     // [n_split_tiles * s * 2] slots of 8 * ws_acc_f4 fp32
    int32_t* counters;             // [n_split_tiles * 2] arrival counters, zero between launches
};

// Early hand-back of ONE expert's slot (ef_internal.h, EfEarly): group 0 of the table is the hit whose slot the visit's first
// pending copy will overwrite -- a decode-sized expert: ONE short token tile.  Its units are the first tickets of the launch:
// [0, e1) its GEMM1 units, [e1, e1 + e2) its GEMM2 units (split s ways along K like a tail when split0), ahead of every unit
// of the other groups, whose phases are planned and ordered as if group 0 were not in the wave.  Still deadlock-free: its
// GEMM2 units depend only on lower tickets, which never wait.  Each of its GEMM2 units adds its k-blocks to *flag once its MMAs
// have completed, i.e. once nothing of the unit reads the slot any more; the copy stream waits for the sum
// (cuStreamWaitValue32), not for the end of the launch.
struct EarlyArgs {
    int32_t e1, e2;         // e1 == 0: off
    uint32_t* flag;
    int32_t split0, tail0;  // split0: group 0's GEMM2 tiles are split p1.s ways, workspace slots / counters from index tail0 on
};

struct Tile {
    int phase;           // 0: GEMM1 unit, 1: GEMM2 unit
    int a_row, c_row;    // first token row in the A tensor / in the output
    int rows_valid;      // tokens of this tile (1..256)
    int n_mma;           // rows_valid rounded up to the MMA N granularity (16)
    int is_long;         // > 128 tokens: takes the whole TMEM
    int n_pair, slot;    // n_pair: the pair's two adjacent weight tiles are 2 * n_pair + cluster rank
    int kb0, kb1;        // k-block range of this unit
    int tail, split_j;   // index among the split tiles (-1: whole tile) and which K part this unit is
    int tid;             // token-tile id inside the launch: index of the "h rows ready" counter
    int g;               // group (index into the wave table)
};

// Token tiling of a group.  A tile narrower than ~170 tokens costs as much per k-block as a 170-token one (its 32 KB
// weight stage has to be filled either way), so with long K loops a group of 257..4096 rows is cut into
// ceil(rows / 256) BALANCED tiles of b = ceil16(rows / tiles) rows instead of full 256-row tiles plus a small remainder
// (593 rows: 208 + 208 + 177, not 256 + 256 + 81): measured +5 % / +3 % on GEMM1 / GEMM2 of the Mixtral shape.  With a
// short K loop (the many-expert shapes) one more 129..256-token tile has a fixed cost -- its epilogue is not overlapped,
// it owns all of TMEM: while the TMEM hand-over still paid a cluster-scope release that outweighed the balance (-2 % /
// -6 %) and those shapes kept 256-row tiles + remainder (kBalancedMinK = 3072); with the relaxed hand-over balanced
// tiles win there too (cfg 4, all experts resident: 389 -> 385 us), so every shape is balanced now.
// Both GEMMs of a wave use the SAME tiling, so that a GEMM2 unit depends on exactly one token tile of GEMM1.  Tiles
// 0 .. n-2 hold b rows, the last one what is left; it is "short" (<= 128 tokens, half of TMEM) or "long".
constexpr int kBalancedMinK = 0;
__device__ __host__ __forceinline__ int group_tile_rows(int rows, bool balanced) {
    const int n = (rows + BT - 1) / BT;
    if (!balanced || n < 2 || n > 16) return BT;
    const int b = (((rows + n - 1) / n) + 15) & ~15;
    return ((n - 1) * b < rows) ? b : BT;
}
// (the b == BT paths are shifts and masks: the kernel prologue walks up to 64 groups in one thread)
__device__ __host__ __forceinline__ int group_long_tiles(int rows, bool balanced) {
    const int b = group_tile_rows(rows, balanced);
    if (b == BT) return rows / BT + ((rows % BT) > 128 ? 1 : 0);
    return rows / b + ((rows % b) > 128 ? 1 : 0);
}
__device__ __host__ __forceinline__ int group_has_short(int rows, bool balanced) {
    const int b = group_tile_rows(rows, balanced);
    const int r = (b == BT) ? rows % BT : rows % b;
    return (r > 0 && r <= 128) ? 1 : 0;
}

__device__ __forceinline__ Tile decode_tile(const EfWaveTable& tab, const SmemCtl* ctl, int unit, const PhaseArgs& p0,
                                            const PhaseArgs& p1, const EarlyArgs& early) {
    Tile t;
    t.tail = -1; t.split_j = 0;
    int g = 0, j = 0;
    if (unit < early.e1 + early.e2) {
        // group 0's single short tile (early hand-back): its GEMM1 units, then its GEMM2 units
        t.phase = unit >= early.e1 ? 1 : 0;
        const PhaseArgs& p = t.phase ? p1 : p0;
        t.kb0 = 0; t.kb1 = p.KB;
        t.n_pair = unit - (t.phase ? early.e1 : 0);
        if (t.phase == 1 && early.split0) {
            const int k = t.n_pair;
            t.n_pair = k / p.s;
            t.split_j = k - t.n_pair * p.s;
            t.tail = early.tail0 + t.n_pair;
            t.kb0 = (t.split_j * p.KB) / p.s;
            t.kb1 = ((t.split_j + 1) * p.KB) / p.s;
        }
        t.is_long = 0;
    } else {
        // the other groups (all groups when there is no early group): tickets in canonical order, all GEMM1 units, then all GEMM2 units
        const int skip = early.e1 > 0 ? 1 : 0;      // group 0 is not part of this order
        unit -= early.e1 + early.e2;
        t.phase = unit >= p0.total ? 1 : 0;
        const PhaseArgs& p = t.phase ? p1 : p0;
        const int u = unit - (t.phase ? p0.total : 0);
        int tile = u;
        t.kb0 = 0; t.kb1 = p.KB;
        if (u >= p.n_plain) {
            const int v = u - p.n_plain;
            t.tail = v / p.s;
            t.split_j = v - t.tail * p.s;
            tile = p.n_plain + t.tail;
            t.kb0 = (t.split_j * p.KB) / p.s;
            t.kb1 = ((t.split_j + 1) * p.KB) / p.s;
        }
        // Ticket order inside a phase: long (129..256-token) tiles are tensor-bound, short ones are bound by streaming their
        // weight tile, so a launch with many short tiles (many-expert prefill) spreads them evenly among the long ones --
        // both kinds are then in flight on different SMs at the same time -- and keeps only the last `tail_short` short
        // tiles for the end of the list, where small units even out the finish (and where the split-K tail lives).
        const int npn = p.n_pairs_n;
        const int skip_short = skip * npn;          // the early group's tile is short and the first of the short tiles
        const int total_long = ctl->tl[tab.n] * npn, total_short = ctl->tsh[tab.n] * npn - skip_short;
        const int tail_short = min(total_short, (int)gridDim.x / 4);
        const int spread = total_short - tail_short, first = total_long + spread;
        bool is_short;
        if (tile >= first) {
            is_short = true;
            tile = spread + (tile - first);
        } else {
            const int sb = (int)(((long long)tile * spread) / first), sb1 = (int)(((long long)(tile + 1) * spread) / first);
            is_short = sb1 > sb;
            tile = is_short ? sb : tile - sb;
        }
        if (!is_short) {
            while (tile >= ctl->tl[g + 1] * npn) ++g;
            const int local = tile - ctl->tl[g] * npn;
            const int nl = ctl->g_long[g];
            t.n_pair = local / nl;                  // n-major inside a group: the token tiles that share a weight tile are
            j = local - t.n_pair * nl;              // claimed back to back and hit L2
            t.is_long = 1;
        } else {
            tile += skip_short;
            while (tile >= ctl->tsh[g + 1] * npn) ++g;
            t.n_pair = tile - ctl->tsh[g] * npn;
            j = ctl->g_long[g];
            t.is_long = 0;
        }
    }
    const int row_off = j * ctl->g_tile_rows[g];
    t.tid = ctl->tl[g] + ctl->tsh[g] + j;
    t.rows_valid = min(tab.g[g].rows - row_off, (int)ctl->g_tile_rows[g]);
    t.n_mma = (t.rows_valid + 15) & ~15;
    t.a_row = (t.phase ? tab.g[g].h_row0 : tab.g[g].x_row0) + row_off;
    t.c_row = (t.phase ? tab.g[g].y_row0 : tab.g[g].h_row0) + row_off;
    t.slot = tab.g[g].slot;
    t.g = g;
    return t;
}

// "h rows of token tile tid are complete": GEMM1 units add 1 per weight tile stored, GEMM2 producers wait for all of them.
__device__ __forceinline__ void signal_ready(int32_t* cnt) {
    asm volatile("fence.proxy.async;" ::: "memory");
    asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(cnt) : "memory");
}
__device__ __forceinline__ void wait_ready(const int32_t* cnt, int need) {
    // The GEMM1 units this waits for were all claimed before the first GEMM2 ticket was handed out, by CTAs that never wait
    // themselves, so the wait is bounded by one unit's duration.  A signal that never comes would be a bug in this file:
    // after 10 s of wall time (globaltimer; robust against slow clocks, preemption and profilers' replays) the kernel
    // traps -- a sticky CUDA error at the C ABI -- instead of hanging the device.
    int v = 0;
    unsigned long long t0 = 0;
    for (unsigned spins = 0;; ++spins) {
        asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(cnt) : "memory");
        if (v >= need) break;
        __nanosleep(100);
        if ((spins & 1023u) == 1023u) {
            unsigned long long t;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
            if (t0 == 0) t0 = t;
            else if (t - t0 > 10000000000ull) __trap();
        }
    }
    asm volatile("fence.proxy.async;" ::: "memory");                // the rows were written through the generic proxy; TMA reads them
}

// Epilogue of one unit for the 8 epilogue warps of one CTA.  kEpi: 0 plain (GEMM2), 1 SwiGLU (gated GEMM1: accumulator 0
// = 128 gate rows, accumulator 1 = the matching up rows -> 128 output columns per weight tile), 2 ReLU (non-gated GEMM1
// of Switch-style experts, R30); for 0 and 2 accumulators 0 / 1 = output columns [256 n, +128) / [256 n + 128, +128).
template <int kEpi>
__device__ __forceinline__ void epilogue_unit(const Tile& t, const PhaseArgs& p, SmemCtl* ctl, uint8_t* stg_base, uint32_t tmem_base,
                                              uint32_t rank, int warp, int lane, int b0, int nb, int32_t* ready, bool do_signal) {
    constexpr bool kSwiglu = kEpi == 1;
    constexpr bool kRelu = kEpi == 2;
    const int q = warp & 3;
    const int part = (warp - 4) >> 2;
    const int lane128 = q * 32 + lane;            // accumulator lane = weight row inside the 128-row block
    const int n_tile = 2 * t.n_pair + (int)rank;
    const bool tile_ok = n_tile < p.n_tiles_n;    // false: the odd last weight tile's idle partner
    const bool split = t.tail >= 0;
    const size_t slot_floats = (size_t)8 * p.ws_acc_f4;
    float* ws_mine = split ? p.ws + (((size_t)t.tail * p.s + t.split_j) * 2 + rank) * slot_floats : nullptr;
    uint16_t* __restrict__ C = p.C;
    const int ldc = p.ldc, n_cols = p.n_cols;
    const uint32_t tb0 = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(b0 * 256);
    const uint32_t tb1 = tb0 + (t.is_long ? 256u : 128u);
    const int n_chunks = tile_ok ? (t.rows_valid + 31) >> 5 : 0;
    const int col0 = kSwiglu ? n_tile * ACC_M : n_tile * BW;      // first output column of accumulator 0
    uint8_t* stg = stg_base + part * STG_BYTES;
    // stmatrix row address of this thread: block i = lane / 8 (tokens 8i..8i+7), row lane % 8, + feature offset
    const uint32_t st_row = smem_u32(stg) + (uint32_t)(lane * STG_LD + q * 64);
#pragma unroll 1
    for (int c = part; c < n_chunks; c += 2) {
        const int n_rows = min(32, t.rows_valid - c * 32);
        if (split) {
            uint32_t a0[32];
            tc_ld32(tb0 + c * 32, a0);
            tc_wait_ld();
            ws_store32(ws_mine, p.ws_acc_f4, 0, c, lane128, a0);
            tc_ld32(tb1 + c * 32, a0);
            tc_wait_ld();
            ws_store32(ws_mine, p.ws_acc_f4, 1, c, lane128, a0);
            continue;
        }
#pragma unroll 1
        for (int acc = 0; acc < (kSwiglu ? 1 : 2); ++acc) {
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const uint32_t lane_off = (uint32_t)(hh * 16) << 16;
                uint32_t r[8];
                if (kSwiglu) {
                    uint32_t g[16], u[16];
                    tc_ld16x256b_x4(tb0 + lane_off + c * 32, g);
                    tc_ld16x256b_x4(tb1 + lane_off + c * 32, u);
                    tc_wait_ld();
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        r[i] = pack_bf16(silu_mul(__uint_as_float(g[2 * i]), __uint_as_float(u[2 * i])),
                                         silu_mul(__uint_as_float(g[2 * i + 1]), __uint_as_float(u[2 * i + 1])));
                } else {
                    uint32_t v[16];
                    tc_ld16x256b_x4((acc ? tb1 : tb0) + lane_off + c * 32, v);
                    tc_wait_ld();
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        float lo = __uint_as_float(v[2 * i]), hi = __uint_as_float(v[2 * i + 1]);
                        if (kRelu) { lo = fmaxf(lo, 0.f); hi = fmaxf(hi, 0.f); }
                        r[i] = pack_bf16(lo, hi);
                    }
                }
                // r[2j] = lanes 0-7 of this half, r[2j+1] = lanes 8-15; token block j
                stmatrix_x4_trans(st_row + hh * 32, r[0], r[2], r[4], r[6]);
                stmatrix_x4_trans(st_row + hh * 32 + 16, r[1], r[3], r[5], r[7]);
            }
            stage_to_global(stg, C, ldc, (int64_t)t.c_row + c * 32, n_rows, col0 + acc * ACC_M, n_cols, lane128, 2 + part);
        }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0)
        for (int h = 0; h < nb; ++h) mbar_arrive_remote_relaxed(mapa(&ctl->tmem_empty[b0 + h], 0));
    bool stored = !split && tile_ok;              // this CTA has written its part of the output tile
    if (split && tile_ok) {
        // publish the partial, count arrivals; the last unit of the tile reduces all s partials in split order
        __threadfence();
        epi_bar();
        if (threadIdx.x == 4 * 32) {
            int32_t* cnt = p.counters + t.tail * 2 + rank;
            const int old = atomicAdd(cnt, 1);
            const int last = (old == p.s - 1) ? 1 : 0;
            if (last) *cnt = 0;                          // re-arm for the next launch
            ctl->split_last = last;
        }
        epi_bar();
        const bool last = ctl->split_last != 0;          // rewritten only after the next split unit's first barrier
        if (last) {
            __threadfence();
            const float* ws_tile = p.ws + ((size_t)t.tail * p.s * 2 + rank) * slot_floats;
            uint16_t* srow = reinterpret_cast<uint16_t*>(stg) + lane128;           // [token][feature], 2-byte stores
            if (kSwiglu) {
#pragma unroll 1
                for (int c = part; c < n_chunks; c += 2) {
                    const int n_rows = min(32, t.rows_valid - c * 32);
                    uint32_t a0[32], a1[32];
                    ws_sum32(ws_tile, p.ws_acc_f4, p.s, 0, c, lane128, a0);
                    ws_sum32(ws_tile, p.ws_acc_f4, p.s, 1, c, lane128, a1);
#pragma unroll
                    for (int i = 0; i < 32; ++i)
                        srow[i * (STG_LD / 2)] = bf16_bits(silu_mul(__uint_as_float(a0[i]), __uint_as_float(a1[i])));
                    stage_to_global(stg, C, ldc, (int64_t)t.c_row + c * 32, n_rows, col0, n_cols, lane128, 2 + part);
                }
            } else {
                // the two accumulators are independent output columns: the (chunk, accumulator) items alternate between the
                // two warp groups, so a one-chunk decode tile is reduced by both groups at once
#pragma unroll 1
                for (int w = part; w < 2 * n_chunks; w += 2) {
                    const int c = w >> 1, acc = w & 1;
                    const int n_rows = min(32, t.rows_valid - c * 32);
                    uint32_t a0[32];
                    ws_sum32(ws_tile, p.ws_acc_f4, p.s, acc, c, lane128, a0);
#pragma unroll
                    for (int i = 0; i < 32; ++i) {
                        float v = __uint_as_float(a0[i]);
                        if (kRelu) v = fmaxf(v, 0.f);
                        srow[i * (STG_LD / 2)] = bf16_bits(v);
                    }
                    stage_to_global(stg, C, ldc, (int64_t)t.c_row + c * 32, n_rows, col0 + acc * ACC_M, n_cols, lane128, 2 + part);
                }
            }
            stored = true;
        }
    }
    // GEMM1 of a fused wave: tell the GEMM2 units of this token tile that one more weight tile's h columns are in place
    if (do_signal && stored) {
        __threadfence();
        epi_bar();
        if (threadIdx.x == 4 * 32) signal_ready(ready + t.tid);
    }
}

template <bool kReluExperts>     // false: SwiGLU experts (gated GEMM1); true: Switch-style ReLU experts
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
ffn_wave_kernel(const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmH,
                const __grid_constant__ CUtensorMap tmW, const PhaseArgs p0, const PhaseArgs p1, int slot_rowlets,
                int balanced, int n_token_tiles, int32_t* __restrict__ sched /* {tickets, finished CTAs, ready[n_token_tiles]} */,
                long long* __restrict__ kprof, const EarlyArgs early, const __grid_constant__ EfWaveTable tab) {
    extern __shared__ uint8_t smem_raw[];
    KTIME(long long kt_entry; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(kt_entry));)
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* stg_base = smem + (size_t)kStages * STAGE_BYTES;
    SmemCtl* ctl = (SmemCtl*)(stg_base + 2 * STG_BYTES);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const bool leader = rank == 0;
    const int total_tiles = early.e1 + early.e2 + p0.total + p1.total;
    int32_t* ready = sched + 2;
    // a GEMM2 unit waits for the h columns of all real weight tiles of GEMM1 (only when GEMM1 runs in this launch)
    const int ready_need = (p0.total > 0 && p1.total > 0) ? p0.n_tiles_n : 0;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmX) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmH) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmW) : "memory");
    }
    if (warp == 1 && lane == 0) {
        for (int i = 0; i < kStages; ++i) { mbar_init(&ctl->full[i], 1); mbar_init(&ctl->empty[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&ctl->tmem_full[i], 1); mbar_init(&ctl->tmem_empty[i], 2 * kEpiWarps); }
        for (int i = 0; i < kSched; ++i) { mbar_init(&ctl->sched_full[i], 1); mbar_init(&ctl->sched_empty[i], 2 * (1 + kEpiWarps)); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&ctl->tmem_base)), "r"(kTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    if (warp == 3) {
        // per-group token tiling (lanes in parallel), then the exclusive scans of the tile counts (one lane)
        for (int g = lane; g < tab.n; g += 32) {
            const int rows = tab.g[g].rows;
            const int nlg = group_long_tiles(rows, balanced != 0);
            ctl->g_tile_rows[g] = (int16_t)group_tile_rows(rows, balanced != 0);
            ctl->g_long[g] = (int16_t)nlg;
            ctl->tl[g + 1] = nlg;
            ctl->tsh[g + 1] = group_has_short(rows, balanced != 0);
        }
        __syncwarp();
        if (lane == 0) {
            int nl = 0, ns = 0;
            ctl->tl[0] = 0;
            ctl->tsh[0] = 0;
            for (int g = 1; g <= tab.n; ++g) {
                nl += ctl->tl[g];  ctl->tl[g] = nl;
                ns += ctl->tsh[g]; ctl->tsh[g] = ns;
            }
        }
    }
    tc_fence_before();
    cluster_sync();               // barriers of both CTAs are initialised before any remote arrive / multicast commit
    tc_fence_after();
    const uint32_t tmem_base = ctl->tmem_base;

    if (warp == 0) {
        // ===== tile scheduler (leader) + TMA producer (both) =====
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int it = 0;; ++it) {
                const int ss = it % kSched;
                int tile;
                if (leader) {
                    mbar_wait_cluster(&ctl->sched_empty[ss], ((it / kSched) & 1) ^ 1);
                    tile = atomicAdd(sched, 1);
                    ctl->sched_tile[ss] = tile;
                    mbar_arrive(&ctl->sched_full[ss]);                       // release.cta: local waiters
                    // the peer's copy and its barrier's 4 transaction bytes in one st.async (its producer lane arms them)
                    st_async_u32(mapa(&ctl->sched_tile[ss], 1), (uint32_t)tile, mapa(&ctl->sched_full[ss], 1));
                } else {
                    mbar_expect_tx(&ctl->sched_full[ss], 4);                 // this lap's arrival + the leader's 4 bytes
                    mbar_wait_cluster(&ctl->sched_full[ss], (it / kSched) & 1);
                    tile = ctl->sched_tile[ss];
                    mbar_arrive_remote_relaxed_after(mapa(&ctl->sched_empty[ss], 0), tile);
                }
                if (tile >= total_tiles) break;
                const Tile t = decode_tile(tab, ctl, tile, p0, p1, early);
                const PhaseArgs& p = t.phase ? p1 : p0;
                const CUtensorMap* tmA = t.phase ? &tmH : &tmX;
                const int half = t.n_mma >> 1;                               // token rows this CTA stages
                const int n_box = (half + XBOX - 1) / XBOX;
                const uint32_t bytes = (uint32_t)(W_BYTES + n_box * XBOX_BYTES);
                // weight tile -> rowlet coordinates in the arena (tiled layout, ef_internal.h): a k-block of the tile is
                // h_t contiguous rowlets.  The odd last pair's partner has no weight tile: it stages only its half of the
                // tokens (the MMA multiplies whatever its weight stage holds; its lanes are never stored).  A short last
                // tile's box runs on into the next k-block's rowlets (lanes >= h_t, never stored either)
                const bool peer_idle = 2 * t.n_pair + 1 >= p.n_tiles_n;
                const bool w_idle = peer_idle && rank == 1;
                const int w_tile = w_idle ? 0 : 2 * t.n_pair + (int)rank;
                const int h_t = min(BW, p.w_rows - w_tile * BW);
                const int w_rowlet0 = t.slot * slot_rowlets + p.base_rowlet + w_tile * BW * p.KB;
                const int x_row = t.a_row + (int)rank * half;
                bool must_wait = t.phase == 1 && ready_need > 0;
                for (int kb = t.kb0; kb < t.kb1; ++kb) {
                    mbar_wait(&ctl->empty[stage], phase ^ 1);
                    uint8_t* sw = smem + (size_t)stage * STAGE_BYTES;
                    if (leader) mbar_expect_tx(&ctl->full[stage], 2 * bytes - (peer_idle ? (uint32_t)W_BYTES : 0u));  // both CTAs' boxes land here
                    const uint32_t bar = mapa(&ctl->full[stage], 0);
                    if (!w_idle) tma_load_2d(sw, &tmW, bar, 0, w_rowlet0 + kb * h_t);
                    if (must_wait) {
                        // the weights do not depend on GEMM1: their box is already on its way while this lane waits for
                        // the h rows of its token tile (written by the GEMM1 units of this same launch)
                        wait_ready(ready + t.tid, ready_need);
                        must_wait = false;
                    }
                    for (int j = 0; j < n_box; ++j)
                        tma_load_2d(sw + W_BYTES + j * XBOX_BYTES, tmA, bar, kb * BK, x_row + j * XBOX);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (leader CTA only) =====
        // The WHOLE warp runs this loop in step and one elected lane issues: every operand of a tcgen05 instruction is then a
        // warp-uniform value the compiler keeps in uniform registers (values read from shared memory are made uniform with a
        // shuffle from lane 0).  Issued from inside an `if (lane == 0)` region instead, each tcgen05.mma costs a loop of
        // ELECT + 7 R2UR.BROADCAST (~74 clocks): more than the tensor time of an MMA of <= 128 tokens.
        if (leader) {
            int stage = 0; uint32_t phase = 0;
            int buf = 0; uint32_t bphase = 0;          // bit b = phase of TMEM half b
            const uint32_t tmem_u = (uint32_t)__shfl_sync(0xffffffffu, (int)tmem_base, 0);
            const uint32_t smem_u = (uint32_t)__shfl_sync(0xffffffffu, (int)smem_u32(smem), 0);
            KPROF(long long kp_t0 = clock64(); long long kp_sched = 0, kp_tmem = 0, kp_full = 0; int kp_units = 0;)
            KTIME(long long kt[5] = {kt_entry, 0, 0, 0, 0}; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(kt[1]));)
            for (int it = 0;; ++it) {
                const int ss = it % kSched;
                KPROF(long long kp_a = clock64();)
                mbar_wait(&ctl->sched_full[ss], (it / kSched) & 1);
                KPROF(kp_sched += clock64() - kp_a;)
                const int tile = __shfl_sync(0xffffffffu, ctl->sched_tile[ss], 0);   // (also: every lane has read the slot)
                if (lane == 0) mbar_arrive(&ctl->sched_empty[ss]);
                if (tile >= total_tiles) break;
                KPROF(++kp_units;)
                const Tile t = decode_tile(tab, ctl, tile, p0, p1, early);
                const int is_long = __shfl_sync(0xffffffffu, t.is_long, 0), n_mma = __shfl_sync(0xffffffffu, t.n_mma, 0);
                const int kb0 = __shfl_sync(0xffffffffu, t.kb0, 0), kb1 = __shfl_sync(0xffffffffu, t.kb1, 0);
                const int b0 = is_long ? 0 : buf, nb = is_long ? 2 : 1;
                KPROF(long long kp_b = clock64();)
                for (int h = 0; h < nb; ++h) mbar_wait_cluster(&ctl->tmem_empty[b0 + h], ((bphase >> (b0 + h)) & 1u) ^ 1u);
                KPROF(kp_tmem += clock64() - kp_b;)
                tc_fence_after();
                const uint32_t d0 = tmem_u + (uint32_t)(b0 * 256);
                const uint32_t d1 = d0 + (is_long ? 256u : 128u);
                const uint32_t idesc = make_idesc(n_mma);
                for (int kb = kb0; kb < kb1; ++kb) {
                    KPROF(long long kp_c = clock64();)
                    mbar_wait(&ctl->full[stage], phase);
                    KPROF(kp_full += clock64() - kp_c;)
                    KTIME(if (t.phase == 1 && !kt[3]) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(kt[3]));)
                    tc_fence_after();
                    const uint32_t sw = smem_u + (uint32_t)(stage * STAGE_BYTES);
                    const uint32_t sx = sw + W_BYTES;
                    if (elect_one()) {
#pragma unroll
                        for (int k = 0; k < BK / 16; ++k) {
                            const uint64_t xd = smem_desc(sx + k * 32);
                            const uint32_t acc = (kb > kb0 || k > 0) ? 1u : 0u;
                            tc_mma(d0, smem_desc(sw + k * 32), xd, idesc, acc);
                            tc_mma(d1, smem_desc(sw + ACC_M * BK * 2 + k * 32), xd, idesc, acc);
                        }
                        tc_commit(&ctl->empty[stage]);    // frees the smem stage in both CTAs once these MMAs have read it
                    }
                    __syncwarp();
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
                if (elect_one())
                    for (int h = 0; h < nb; ++h) tc_commit(&ctl->tmem_full[b0 + h]);
                __syncwarp();
                for (int h = 0; h < nb; ++h) bphase ^= 1u << (b0 + h);
                buf = is_long ? 0 : (b0 ^ 1);
                KTIME(asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(kt[t.phase == 0 ? 2 : 4]));)
            }
            KTIME(if (kprof && lane == 0) { long long* o = kprof + (size_t)(blockIdx.x >> 1) * 5; for (int i = 0; i < 5; ++i) o[i] = kt[i]; kprof = nullptr; })
            KPROF(if (kprof && lane == 0) {
                long long* o = kprof + (size_t)(blockIdx.x >> 1) * 5;
                o[0] = clock64() - kp_t0; o[1] = kp_sched; o[2] = kp_tmem; o[3] = kp_full; o[4] = kp_units;
            })
        }
    } else if (warp >= 4) {
        // ===== epilogue: warps w and w+4 share TMEM lane quarter (w % 4) and take alternate 32-token chunks =====
        int buf = 0; uint32_t bphase = 0;
        for (int it = 0;; ++it) {
            const int ss = it % kSched;
            mbar_wait_cluster(&ctl->sched_full[ss], (it / kSched) & 1);
            const int tile = ctl->sched_tile[ss];
            __syncwarp();
            if (lane == 0) mbar_arrive_remote_relaxed_after(mapa(&ctl->sched_empty[ss], 0), tile);
            if (tile >= total_tiles) break;
            const Tile t = decode_tile(tab, ctl, tile, p0, p1, early);
            const int b0 = t.is_long ? 0 : buf, nb = t.is_long ? 2 : 1;
            for (int h = 0; h < nb; ++h) {
                mbar_wait(&ctl->tmem_full[b0 + h], (bphase >> (b0 + h)) & 1u);
                bphase ^= 1u << (b0 + h);
            }
            tc_fence_after();
            // the unit's MMAs have completed: neither CTA's stages of it are read any more (early hand-back, see EarlyArgs)
            if (early.e1 > 0 && t.phase == 1 && t.g == 0 && leader && threadIdx.x == 4 * 32)
                asm volatile("red.relaxed.gpu.global.add.u32 [%0], %1;" ::"l"(early.flag), "r"((uint32_t)(t.kb1 - t.kb0)) : "memory");
            if (t.phase == 0)
                epilogue_unit<kReluExperts ? 2 : 1>(t, p0, ctl, stg_base, tmem_base, rank, warp, lane, b0, nb, ready, ready_need > 0);
            else
                epilogue_unit<0>(t, p1, ctl, stg_base, tmem_base, rank, warp, lane, b0, nb, ready, false);
            buf = t.is_long ? 0 : (b0 ^ 1);
        }
    }

    tc_fence_before();
    cluster_sync();               // the peer's TMEM / shared memory / barriers stay alive until both CTAs are done
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
    }
    KTIME(if (threadIdx.x == 0 && kprof) { long long te; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(te)); kprof[(size_t)(148 / 2) * 5 + blockIdx.x] = te; })
    // the last CTA to finish re-arms the scheduler words and the ready counters for the launch that reuses them (every
    // leader has drawn its terminal ticket and every GEMM2 producer has seen its counter by now)
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(sched + 1, 1) == (int)gridDim.x - 1) {
            for (int i = 0; i < n_token_tiles; ++i) ready[i] = 0;
            sched[0] = 0; sched[1] = 0;
        }
    }
}

// ---- host side -------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// 2-D bf16 [rows, K] row-major, box 64 x 64 token rows, 128-byte swizzle
int32_t make_map_2d(ef_ctx* ctx, CUtensorMap* tm, const void* base, int64_t rows, int64_t K) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return ef_fail(ctx, EF_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)K * 2};
    cuuint32_t box[2] = {BK, XBOX};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ef_fail(ctx, EF_ERR_CUDA, "cuTensorMapEncodeTiled(2d) failed: %d", (int)r);
    return EF_OK;
}

// the whole arena as rowlets: 2-D bf16 [total rowlets, 64], box 64 x 256 = one k-block of one weight tile (32 KB, contiguous)
int32_t make_map_arena(ef_ctx* ctx, CUtensorMap* tm, const void* base) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return ef_fail(ctx, EF_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const int64_t rowlets = (int64_t)ctx->n_arena_slots * (ctx->W / (EF_ROWLET * 2));
    if (rowlets + BW > INT32_MAX) return ef_fail(ctx, EF_ERR_UNSUPPORTED, "slot arena too large for 32-bit rowlet coordinates");
    cuuint64_t dims[2] = {(cuuint64_t)EF_ROWLET, (cuuint64_t)rowlets};
    cuuint64_t strides[1] = {(cuuint64_t)EF_ROWLET * 2};
    cuuint32_t box[2] = {BK, BW};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ef_fail(ctx, EF_ERR_CUDA, "cuTensorMapEncodeTiled(arena) failed: %d", (int)r);
    return EF_OK;
}

// per-launch scheduler block {ticket counter, finished CTAs, ready[n_token_tiles]}; the kernel zeroes it again when it
// ends, and the blocks are carved out of a ring that is far longer than anything that can be in flight on one stream
int32_t* next_sched(ef_ctx* ctx, int n_words) {
    if (ctx->sched_next + n_words > EF_SCHED_WORDS) ctx->sched_next = 0;
    int32_t* p = ctx->sched_words + ctx->sched_next;
    ctx->sched_next += n_words;
    return p;
}

// Tail split-K plan for one phase: `tiles` tickets in scheduler order with `n_short` short ones at the end, G CTA pairs,
// KB k-blocks per tile.  Costs are in k-block times of a 256-row tile (1024 tensor cycles): a whole tail tile holds
// an SM for KB (KB/2 if short) of them; a split unit adds a partial write and the finaliser reads s partials
// (~0.03 per valid row each, from the measured ~50 GB/s per-SM global bandwidth, and never less than a dependent
// round trip each).
struct SplitPlan { int n_plain, n_tail, s; };

SplitPlan plan_split(const ef_ctx* ctx, int tiles, int n_short, int G, int KB, double avg_rows, int max_units) {
    SplitPlan p{tiles, 0, 1};
    if (ctx->splitk_mode == 1 || tiles == 0) return p;
    int r = tiles % G;
    if (tiles < G) r = tiles;
    if (ctx->splitk_mode >= 2) {                       // forced (tests): split every tile
        p.s = std::min(ctx->splitk_mode, std::max(1, KB));
        if (p.s < 2) return SplitPlan{tiles, 0, 1};
        p.n_tail = std::min(tiles, max_units / p.s);
        p.n_plain = tiles - p.n_tail;
        return p.n_tail ? p : SplitPlan{tiles, 0, 1};
    }
    if (r == 0) return p;
    const double w = (n_short >= r) ? 0.5 : 1.0;       // the tail is the end of the list: short tiles first
    const double ovh = 0.03 * avg_rows;
    const int smax = std::min(16, KB / 4);
    double best = KB * w;                              // s = 1: one more round of whole tiles
    for (int s = 2; s <= smax; ++s) {
        if (r * s > max_units) break;
        // the finaliser walks the s partials one after the other: bandwidth for wide tiles (ovh per partial), a dependent
        // L2 round trip per partial and accumulator for narrow ones (measured on a 5-token decode tile: ~4 us for s = 5,
        // which turned a 48 us GEMM1 into 68 us -- a decode GEMM1 is not split, its HBM stream is what bounds it)
        const double fin = std::max(ovh * (1 + s), 1.5 * s);
        const double cost = (double)((r * s + G - 1) / G) * (KB * w / s) + 1.0 + fin;
        if (cost < best * 0.9) { best = cost; p.s = s; }
    }
    if (p.s > 1) { p.n_tail = r; p.n_plain = tiles - r; }
    return p;
}

// bytes one phase's TMA loads stage into shared memory (what crosses the L2 -> SM fabric): per token tile and weight-tile
// pair, per k-block, each CTA of the pair pulls its 32 KB weight box (if it has a weight tile) plus the 8 KB token boxes
// covering its half tile
int64_t phase_fill_bytes(const EfWaveTable& tab, bool balanced, int npn, int n_tiles_n, int KB) {
    int64_t per_kb = 0;
    for (int i = 0; i < tab.n; ++i)
        for (int off = 0, b = group_tile_rows(tab.g[i].rows, balanced); off < tab.g[i].rows; off += b) {
            const int n_mma = (std::min(tab.g[i].rows - off, b) + 15) & ~15;
            const int n_box = (n_mma / 2 + XBOX - 1) / XBOX;
            // every CTA of every pair stages its token boxes; one weight box per real weight tile
            per_kb += (int64_t)npn * 2 * n_box * XBOX_BYTES + (int64_t)n_tiles_n * W_BYTES;
        }
    return per_kb * KB;
}

}  // namespace

int32_t efk_ffn_tc_init(ef_ctx* ctx) {
    static_assert(BK == EF_ROWLET && BW == EF_TILE_ROWS, "the packed layout is tiled for this kernel's stage shape");
    int32_t rc = make_map_arena(ctx, &ctx->tm_w, ctx->arena);
    if (rc != EF_OK) return rc;
    if ((rc = make_map_2d(ctx, &ctx->tm_h, ctx->h_ws, ctx->h_rows, ctx->cfg.d_ff)) != EF_OK) return rc;   // fixed for the ctx's life
    EF_CUDA(ctx, cudaFuncSetAttribute(ffn_wave_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
    EF_CUDA(ctx, cudaFuncSetAttribute(ffn_wave_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
    EF_CUDA(ctx, cudaMalloc(&ctx->sched_words, sizeof(int32_t) * EF_SCHED_WORDS));
    EF_CUDA(ctx, cudaMemset(ctx->sched_words, 0, sizeof(int32_t) * EF_SCHED_WORDS));
    // split-K: pair units; each has one workspace slot and one counter per CTA of the pair; one region per GEMM of a wave
    // (splitk_max_units full-size slots per CTA of the pair; a wave of narrower token tiles cuts the same memory into up to
    // 8x as many smaller slots -- a decode wave's tile is one 32-token chunk wide -- hence 8x the arrival counters)
    ctx->splitk_max_units = ctx->n_sms;
    EF_CUDA(ctx, cudaMalloc(&ctx->splitk_ws, sizeof(float) * kSlotFloats * 2 * 2 * (size_t)ctx->splitk_max_units));
    EF_CUDA(ctx, cudaMalloc(&ctx->splitk_counters, sizeof(int32_t) * 2 * 2 * 8 * ctx->splitk_max_units));
    EF_CUDA(ctx, cudaMemset(ctx->splitk_counters, 0, sizeof(int32_t) * 2 * 2 * 8 * ctx->splitk_max_units));
    ctx->tm_ok = true;
    return EF_OK;
}

// One wave: phase bit 0 = GEMM1 (x -> h), bit 1 = GEMM2 (h -> y).  phase == 3 is ONE launch: the GEMM2 units are ticketed
// behind the GEMM1 units and wait, per token tile, for that tile's h columns (see the kernel).
int32_t efk_ffn_tc(ef_ctx* ctx, cudaStream_t st, const void* x, void* y, const EfWaveTable& tab, int phase, EfEarly* early) {
    const int d = ctx->cfg.d_model, f = ctx->cfg.d_ff;
    if (tab.n == 0 || !(phase & 3)) return EF_OK;
    const bool relu = ctx->cfg.expert_kind == 1;
    const bool bal = d >= kBalancedMinK && f >= kBalancedMinK;
    int64_t rows_total = 0, x_rows = 0;
    int mtiles = 0, mshort = 0;       // token tiles of the wave (every group's long tiles plus its short tail tile)
    int widest = 1;                   // rows of the wave's widest token tile
    for (int i = 0; i < tab.n; ++i) {
        rows_total += tab.g[i].rows;
        widest = std::max(widest, std::min(tab.g[i].rows, group_tile_rows(tab.g[i].rows, bal)));
        x_rows = std::max<int64_t>(x_rows, (int64_t)tab.g[i].x_row0 + tab.g[i].rows);
        mtiles += group_long_tiles(tab.g[i].rows, bal) + group_has_short(tab.g[i].rows, bal);
        mshort += group_has_short(tab.g[i].rows, bal);
    }
    const int n_pairs = ctx->n_sms / 2;     // CTA pairs (clusters of 2), one CTA per SM
    const int w1_rows = relu ? f : 2 * f;   // W1 of a non-gated expert, or packed W13
    const int slot_rowlets = (int)(ctx->W / (EF_ROWLET * 2));
    const double avg_rows = (double)rows_total / mtiles;
    PhaseArgs pa[2] = {};
    // GEMM1: 256 packed W13 rows -> 128 h columns; 256 W1 rows -> 256
    const int ntn1 = relu ? (f + BW - 1) / BW : f / 128, ntn2 = (d + BW - 1) / BW;
    // split-K workspace slots are as wide as the wave's widest tile (in 32-token chunks): a decode wave gets 8x the units
    const int chunks = (widest + 31) / 32;
    const int acc_f4 = chunks * 8 * ACC_M;
    const int max_units = ctx->splitk_max_units * (BT / 32) / chunks;
    pa[0] = PhaseArgs{(uint16_t*)ctx->h_ws, f, f, d / BK, ntn1, (ntn1 + 1) / 2, w1_rows, 0, 0, 0, 1, acc_f4, ctx->splitk_ws,
                      ctx->splitk_counters};
    pa[1] = PhaseArgs{(uint16_t*)y, d, d, f / BK, ntn2, (ntn2 + 1) / 2, d, (int)((int64_t)w1_rows * d / EF_ROWLET), 0, 0, 1, acc_f4,
                      ctx->splitk_ws + (size_t)kSlotFloats * 2 * ctx->splitk_max_units,
                      ctx->splitk_counters + 2 * 8 * ctx->splitk_max_units};
    // Early hand-back of group 0's slot (EarlyArgs): group 0 must be ONE short tile (a decode-sized expert: a launch of its
    // own for it is mostly launch, hand-over and tail -- measured on cfg 3: FFN time per step -6 %, step time +0.2 %; an expert
    // of long tiles keeps its own launch, which is an efficient launch and hands the slot back 50-70 us earlier than a wave
    // could, cfg 2: step time +0.3 % for -2 % FFN time).  Its units are ticketed ahead of the wave; the phases of the other
    // groups are planned as if it were not there.
    EarlyArgs ea{0, 0, nullptr, 0, 0};
    bool early_on = false;
    if (early) {
        early->used = false;
        early->add = 0;
        early_on = early->want && phase == 3 && tab.n >= 2 && ctx->splitk_mode <= 1 && ctx->early_flag && tab.g[0].rows <= 128;
    }
    const int skip = early_on ? 1 : 0;
    for (int ph = 0; ph < 2; ++ph) {
        if (!(phase & (1 << ph))) continue;
        PhaseArgs& p = pa[ph];
        const int tiles = (mtiles - skip) * p.n_pairs_n;
        // GEMM1 of a fused wave is followed by GEMM2 units that depend on it: its tail cannot be filled by them when the wave
        // is one token tile deep, so it is split like a launch of its own
        const double avg = early_on ? (double)(rows_total - tab.g[0].rows) / (mtiles - 1) : avg_rows;
        const SplitPlan pl = plan_split(ctx, tiles, (mshort - skip) * p.n_pairs_n, n_pairs, p.KB, avg, max_units);
        p.n_plain = pl.n_plain;
        p.s = pl.s;
        p.total = pl.n_plain + pl.n_tail * pl.s;
    }
    if (early_on) {
        const int t2 = pa[1].n_pairs_n;            // group 0's GEMM2 tiles (pair units)
        ea = EarlyArgs{pa[0].n_pairs_n, t2, ctx->early_flag, 0, 0};
        // split them along K: with the tail's factor if the others' phase has a split tail, else with one that makes about
        // half a round of units -- each unit is then short enough for the slot to come back about as early as from a launch
        // of its own
        if (pa[1].KB >= 8) {
            const int n_tail = (pa[1].total - pa[1].n_plain) / std::max(1, pa[1].s);
            const int s0 = pa[1].s > 1 ? pa[1].s : std::min(std::min(16, pa[1].KB / 4), std::max(2, (n_pairs / 2 + t2 - 1) / t2));
            if (s0 > 1 && (n_tail + t2) * s0 <= max_units) {
                pa[1].s = s0;
                ea.split0 = 1;
                ea.tail0 = n_tail;
                ea.e2 = t2 * s0;
            }
        }
        early->used = true;
        early->add = (uint32_t)(t2 * pa[1].KB);
    }
    if (early && early->dry) return EF_OK;
    const int total = ea.e1 + ea.e2 + pa[0].total + pa[1].total;
    const int grid = 2 * std::min(total, n_pairs);
    if (2 + mtiles > EF_SCHED_WORDS) return ef_fail(ctx, EF_ERR_CAPACITY, "grouped FFN: too many token tiles in one wave");
    if (phase & 1) {
        if (ctx->tm_x_ptr != x || ctx->tm_x_rows != x_rows) {      // the caller's x_perm buffer rarely changes: encode once
            int32_t rc = make_map_2d(ctx, &ctx->tm_x, x, x_rows, d);
            if (rc != EF_OK) return rc;
            ctx->tm_x_ptr = x;
            ctx->tm_x_rows = x_rows;
        }
    } else if (!ctx->tm_x_ptr) {
        ctx->tm_x = ctx->tm_h;                                      // never dereferenced by a GEMM2-only launch
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (ctx->time_kernels) {
        int32_t rc = efk_timing_events(ctx, &e0, &e1);
        if (rc != EF_OK) return rc;
        EF_CUDA(ctx, cudaEventRecord(e0, st));
    }
    int32_t* sched = next_sched(ctx, 2 + mtiles);
    long long* kprof = (phase & 1) ? ctx->kprof1 : ctx->kprof2;
    if (relu)
        ffn_wave_kernel<true><<<grid, kThreads, kSmemBytes, st>>>(ctx->tm_x, ctx->tm_h, ctx->tm_w, pa[0], pa[1], slot_rowlets,
                                                                  bal ? 1 : 0, mtiles, sched, kprof, ea, tab);
    else
        ffn_wave_kernel<false><<<grid, kThreads, kSmemBytes, st>>>(ctx->tm_x, ctx->tm_h, ctx->tm_w, pa[0], pa[1], slot_rowlets,
                                                                   bal ? 1 : 0, mtiles, sched, kprof, ea, tab);
    ctx->launches++;
    EF_CUDA(ctx, cudaGetLastError());
    if (ctx->time_kernels) {
        EF_CUDA(ctx, cudaEventRecord(e1, st));
        ef_ctx::KSpan span{e0, e1, phase & 3, rows_total, tab.n};
        ctx->kspans.push_back(span);
        if (phase & 1) ctx->ktimes.gemm1_fill_bytes += phase_fill_bytes(tab, bal, pa[0].n_pairs_n, pa[0].n_tiles_n, pa[0].KB);
        if (phase & 2) ctx->ktimes.gemm2_fill_bytes += phase_fill_bytes(tab, bal, pa[1].n_pairs_n, pa[1].n_tiles_n, pa[1].KB);
    }
    return EF_OK;
}
