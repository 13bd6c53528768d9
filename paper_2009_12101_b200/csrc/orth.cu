// orth.cu -- the Gram-Schmidt passes over the compressed basis (Fig. 1 lines 5-11 and 17,
// PAPER.md:70-81, 92; the basis is read in its storage format and widened in registers,
// PAPER.md:133, 169-181).  One persistent, TMA-fed kernel in three kinds:
//
//   PASS_DOT      h_c  = sum_i dec(V)[i,c] w_i                                  (S2,  l.5)
//   PASS_UPD      w_i -= sum_c dec(V)[i,c] h_c, ||w||_2, ||w||_inf              (S3,  l.5-6 / l.8-10 / l.17)
//   PASS_UPD_DOT  the update of the first Gram-Schmidt pass AND the inner products of the second
//                 pass, u = dec(V)^T w_new, from ONE read of the basis          (S3 + S2', l.5-8)
//
// Bound: HBM.  Algorithmic bytes per launch: k n B + 8 n (DOT), k n B + 16 n (UPD, UPD_DOT).
// Classical Gram-Schmidt with re-orthogonalisation reads V four times per Arnoldi step (dot, update,
// dot, update); the fused middle pass makes that three, and consecutive passes walk the rows in
// opposite directions so that the tail of one pass is still in the 126 MB L2 when the next begins.
//
// Mapping.  The n rows are cut into tiles of R rows, R*B = F KB per column segment (F = 1, 2, 4: the
// largest that leaves every CTA at least twelve tiles); a tile is the sequence of 32 KB stages
// [32/F columns x F KB].  One persistent CTA per SM takes the tiles t = CTA, CTA + grid, ... (the
// CTAs sweep a contiguous window of the basis together).  A producer warp streams stages into a
// ring of shared memory (up to ~190 KB) with 2D tensor-map TMA boxes [8 columns x 1-2 KB]
// (completion on an mbarrier) and the tile of w into a 4-slot ring, swizzled (wswz); it issues the
// first stages BEFORE griddepcontrol.wait -- the basis is never written by the predecessor kernel.
// Sixteen consumer warps -- two row halves x eight columns -- work on a stage as soon as it lands:
// a warp owns one column of every 8-column chunk and one half of the rows, its lanes own 16-byte
// payload words, so shared-memory reads are conflict free and every warp ends up with the CTA's
// complete partial sums of ITS columns over its rows.  The plain update uses the row-owner mapping
// instead (each thread its own rows, all columns: no cross-warp reduction); the fused kind with
// reduced storage accumulates per column-warp and adds the eight partial row vectors in a fixed
// order through shared memory.  In PASS_UPD_DOT all stages of a row tile stay resident until the
// new w of that tile is known, then are swept a second time while the ring prefetches the next
// tile.  CTA partials go to global memory; the last CTA to finish adds them in a fixed order
// (deterministic, no fp64 atomics), applies the per-vector scales and takes the decisions of
// Fig. 1 lines 7 and 12 on the device.
#include <cuda.h> // CUtensorMap (types only; the encoder is fetched with cudaGetDriverEntryPoint)
#include <type_traits>

#include "device_utils.cuh"

namespace cbg {

enum PassKind : int { PASS_DOT = 0, PASS_UPD = 1, PASS_UPD_DOT = 2 };

constexpr int kColWarps = 8;                            // columns per chunk: one per warp of a row half
constexpr int kConsumerWarps = 2 * kColWarps;           // two row halves
constexpr int kConsumers = kConsumerWarps * 32;
constexpr int kOrthThreads = kConsumers + 32;           // + one producer warp
constexpr int kChunkCols = kColWarps;
constexpr int kMaxChunks = 16;                          // chunks per launch (accumulators live in registers)
constexpr int kMaxRangeCols = kMaxChunks * kChunkCols;  // 128 columns per launch
constexpr int kMaxStages = 8;
constexpr int kWSlots = 4;                              // ring of w tiles: how many row tiles the producer may run ahead
constexpr int kStageBytes = 32 * 1024;                  // 8 columns x 4 KB, 16 x 2 KB or 32 x 1 KB
constexpr int kOrthSmemBytes = 225 * 1024;              // dynamic shared memory of one CTA (one CTA per SM)

struct OrthArgs {
    const void *V;        // payload of the first column of this launch's range
    int64_t ld;
    const double *scales; // [k] sigma_c of the range (fixed-point formats)
    const double *hs;     // [k] update coefficients sigma_c * h_c (UPD kinds)
    const int *d_k;       // if non-null: total column count read on the device (cycle-end x update)
    int c0;               //   ... and the first column of this launch's range within it
    double *w;            // DOT: read; UPD kinds: read and written
    int64_t n;
    int k;                // columns of this launch (<= 128)
    Ctl *ctl;
    double *partials;     // [grid * kLdp]
    double *npart;        // [2 * kMaxGrid]
    double *h_out;        // DOT kinds: h (ORTH1: set; ORTH2 / fused: accumulated)
    double *hs_out;       // DOT kinds: sigma_c * (h_c or u_c), the next update's coefficients
    int mode, step;
    int last_range;       // UPD kinds: the finaliser of this launch publishes the norms
    int nstages;
    int interleave;       // row tiles dealt round-robin to the CTAs (else one contiguous row range per CTA)
    int dir;              // 1: walk the row tiles from the last to the first
};

// 2D tiled TMA copy global -> shared: box [box0 8-byte elements x 8 columns] at element (x, y) of
// the basis seen as a 2D array of 8-byte words [columns][ld * B / 8]; out-of-range parts read as zero.
__device__ __forceinline__ void tma_box_g2s(void *dst_smem, const CUtensorMap *map, int x, int y, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            smem_u32(dst_smem)),
        "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// Barrier among the eight warps of one row half (ids 2 and 3): in the column-mapped update the two
// halves of a tile never exchange data, so they need not wait for each other.
__device__ __forceinline__ void half_bar(int half)
{
    asm volatile("bar.sync %0, %1;" ::"r"(2 + half), "n"(kConsumers / 2) : "memory");
}
__device__ __forceinline__ void consumer_bar()
{
    asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory");
}

// ---- shared-memory map of one CTA -------------------------------------------------------------------
//   [0, 1024)      mbarriers: full[8], empty[8], wfull[4], wempty[4]
//   [1024, 2048)   hs_s[128]   update coefficients of this launch's columns
//   [2048, 4096)   hpart[2][128] per-row-half dot partials of the CTA (epilogue)
//   [4096, ...)    wbuf[4][R]  ring of w tiles
//   then           red[8][R]   per-column-warp partial V h of the current tile (UPD kinds)
//   then           w1buf[R]    the new w of the current tile for the second sweep (UPD kinds)
//   then           stages[ns][8][SEG] ring of column chunks
__host__ __device__ constexpr int orth_fixed_smem(int R, bool has_upd) { return 4096 + kWSlots * 8 * R + (has_upd ? 72 * R : 0); }

template <int FMT, int F> struct Tile {
    using Fm = Fmt<FMT>;
    static constexpr int VEC = Fm::VEC, B = Fm::BYTES;
    static constexpr int SEG = F * 1024;           // bytes of one column segment
    static constexpr int R = SEG / B;              // rows of a tile
    static constexpr int GV = F * VEC;             // rows (doubles) per lane and column
    static constexpr int CPS = 4 / F;              // chunks per stage: a stage is always 32 columns-KB
    static constexpr int STAGE_COLS = CPS * kChunkCols;
    static constexpr int STAGE = STAGE_COLS * SEG; // bytes of one stage (32 KB)
    static constexpr int WORDS_HALF = F * 32;      // 16-byte words per column and row half
    // TMA boxes: 8 columns x min(SEG, 2 KB); a stage is 4 (F = 1) or 2 (F = 2, 4) boxes.  For
    // F = 4 the two boxes of a stage are the two 2 KB halves of the same 8 columns.
    static constexpr int BOX_INNER = (F == 1 ? 1024 : 2048);
    static constexpr int BOX_BYTES = kChunkCols * BOX_INNER;
    static constexpr int BOXES = STAGE / BOX_BYTES;
    // address of 16-byte word wi (0 .. SEG/16) of column lc (0 .. STAGE_COLS) of a stage
    static __device__ __forceinline__ const unsigned char *word_ptr(const unsigned char *stage, int lc, int wi)
    {
        if constexpr (F == 4) return stage + (wi >> 7) * BOX_BYTES + lc * BOX_INNER + (wi & 127) * 16;
        else return stage + lc * SEG + wi * 16;
    }
};

// Inner product of one decoded payload word with the matching rows of w: two independent chains of
// VEC/2 FMAs (a single chain of 8 dependent fp64 FMAs per word starves the pipe at 4 warps per scheduler).
template <int VEC> __device__ __forceinline__ double word_dot(const double (&d)[VEC], const double *w)
{
    double t0 = d[0] * w[0], t1 = d[1] * w[1];
#pragma unroll
    for (int v = 2; v < VEC; v += 2) {
        t0 = fma(d[v], w[v], t0);
        t1 = fma(d[v + 1], w[v + 1], t1);
    }
    return t0 + t1;
}

// The payload words of this lane in NC consecutive chunks of a stage (its column `cw` of each chunk,
// F words per column): ALL loads are issued first, then every word is widened and handed to
// `fn(i, f, d)` (chunk, word, VEC values / PRE^2).  With the loads up front and no branch in between
// the NC * F independent decode + FMA chains interleave; one word at a time left every warp with a
// single chain and the SM (4 warps per scheduler) half idle.  RAGGED: rows at or beyond `rows` are
// forced to zero (the payload there is stale shared memory or padding and may decode to NaN).
template <int FMT, int F, int NC, bool RAGGED, class Fn>
__device__ __forceinline__ void for_stage_words(const unsigned char *stage, int cw, int wi0, int rows, Fn &&fn)
{
    using T = Tile<FMT, F>;
    uint4 raw[NC][F];
#pragma unroll
    for (int i = 0; i < NC; ++i)
#pragma unroll
        for (int f = 0; f < F; ++f) {
            const int wi = wi0 + f * 32;
            if (RAGGED && wi * T::VEC >= rows) raw[i][f] = make_uint4(0u, 0u, 0u, 0u);
            else raw[i][f] = *reinterpret_cast<const uint4 *>(T::word_ptr(stage, i * kChunkCols + cw, wi));
        }
#pragma unroll
    for (int i = 0; i < NC; ++i)
#pragma unroll
        for (int f = 0; f < F; ++f) {
            double d[T::VEC];
            T::Fm::decode(raw[i][f], d);
            if (RAGGED) {
                const int wi = wi0 + f * 32;
#pragma unroll
                for (int v = 0; v < T::VEC; ++v)
                    if (wi * T::VEC + v >= rows) d[v] = 0.0;
            }
            fn(i, f, d);
        }
}

// Dispatch on the number of chunks of the stage in which this warp's column exists (nv = CPS for
// every stage but the last of a row tile).
template <int FMT, int F, bool RAGGED, class Fn>
__device__ __forceinline__ void for_valid_chunks(int nv, const unsigned char *stage, int cw, int wi0, int rows, Fn &&fn)
{
    constexpr int CPS = Tile<FMT, F>::CPS;
    if (nv >= CPS) {
        for_stage_words<FMT, F, CPS, RAGGED>(stage, cw, wi0, rows, fn);
    } else if constexpr (CPS >= 2) {
        if (nv == 1) for_stage_words<FMT, F, 1, RAGGED>(stage, cw, wi0, rows, fn);
        if constexpr (CPS == 4) {
            if (nv == 2) for_stage_words<FMT, F, 2, RAGGED>(stage, cw, wi0, rows, fn);
            if (nv == 3) for_stage_words<FMT, F, 3, RAGGED>(stage, cw, wi0, rows, fn);
        }
    }
}

// Location of a row of a w tile in shared memory.  A lane owns 16-byte payload words, i.e. VEC
// consecutive rows = VEC * 8 bytes of w: read linearly, the lanes of a warp are 32 or 64 bytes apart
// and every 128-bit load is a 2- or 4-way bank conflict (measured: ~1 us per tile for the 16-bit
// formats, all sixteen warps stalled -- the whole k-independent cost of a pass).  The tiles are
// therefore stored with the TMA 32-byte / 64-byte swizzle (16-byte chunk index XOR address bits
// 7.. ), which spreads the lanes of a quarter warp over all eight 16-byte bank groups.  fp64
// (16 bytes of w per word) needs none.
template <int VEC> __device__ __forceinline__ int wswz(uint32_t base_saddr, int idx) // idx: row of the tile at shared address base_saddr
{
    if constexpr (VEC == 2) return idx;
    const uint32_t a = base_saddr + (uint32_t)idx * 8u;
    return idx ^ (int)(((a >> 7) & (VEC == 8 ? 3u : 1u)) << 1); // 16-byte chunk index XOR address bits 7..: two doubles per chunk
}

// ---- row-owner mapping of the update -----------------------------------------------------------------
// Each of the 512 consumer threads owns SEG / 512 = 2 F bytes of every column segment -- one or two
// whole entries when 2 F >= B -- i.e. its own rows of the tile: the sum over ALL columns stays in the
// thread (no partial row vectors through shared memory, no CTA barrier for the reduction), every
// thread works on every column whatever k is, and the new w leaves the thread that computed it.
// Entries go through the conversion pipe here (one instruction each; true values, unscaled
// coefficients); the dot sweeps keep the integer widening.
// Used for the plain update and for the fused kind with fp64 storage; the fused kind with reduced
// storage is faster with the column mapping (measured, fp16 k = 100, n = 4.2e6: 261 vs 289 us -- one
// 2-byte shared-memory load per entry costs more than the reduction it saves).
template <int FMT, int F, int KIND> __host__ __device__ constexpr bool upd_rowmap()
{
    return 2 * F >= Fmt<FMT>::BYTES && (KIND == PASS_UPD || FMT == CBGMRES_FP64);
}

__device__ __forceinline__ void half2_cvt(unsigned w, double &lo, double &hi) // F2F.F64.F16 takes either half of a register
{
    asm("{.reg .b16 l, h; mov.b32 {l, h}, %2; cvt.f64.f16 %0, l; cvt.f64.f16 %1, h;}" : "=d"(lo), "=d"(hi) : "r"(w));
}
__device__ __forceinline__ void i16x2_cvt(unsigned w, double &lo, double &hi)
{
    asm("{.reg .b16 l, h; mov.b32 {l, h}, %2; cvt.rn.f64.s16 %0, l; cvt.rn.f64.s16 %1, h;}" : "=d"(lo), "=d"(hi) : "r"(w));
}
template <int FMT, int UB> struct Unit; // UB payload bytes -> EU = UB / B doubles
template <> struct Unit<CBGMRES_FP64, 8> {
    static constexpr int EU = 1;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[1]) { d[0] = *reinterpret_cast<const double *>(p); }
};
template <> struct Unit<CBGMRES_FP32, 4> {
    static constexpr int EU = 1;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[1]) { d[0] = (double)*reinterpret_cast<const float *>(p); }
};
template <> struct Unit<CBGMRES_FP32, 8> {
    static constexpr int EU = 2;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[2])
    {
        const float2 f = *reinterpret_cast<const float2 *>(p);
        d[0] = (double)f.x;
        d[1] = (double)f.y;
    }
};
template <> struct Unit<CBGMRES_INT32, 4> {
    static constexpr int EU = 1;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[1]) { d[0] = (double)*reinterpret_cast<const int *>(p); }
};
template <> struct Unit<CBGMRES_INT32, 8> {
    static constexpr int EU = 2;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[2])
    {
        const int2 q = *reinterpret_cast<const int2 *>(p);
        d[0] = (double)q.x;
        d[1] = (double)q.y;
    }
};
template <> struct Unit<CBGMRES_FP16, 2> {
    static constexpr int EU = 1;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[1])
    {
        const unsigned short h = *reinterpret_cast<const unsigned short *>(p);
        asm("cvt.f64.f16 %0, %1;" : "=d"(d[0]) : "h"(h));
    }
};
template <> struct Unit<CBGMRES_FP16, 4> {
    static constexpr int EU = 2;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[2]) { half2_cvt(*reinterpret_cast<const unsigned *>(p), d[0], d[1]); }
};
template <> struct Unit<CBGMRES_INT16, 2> {
    static constexpr int EU = 1;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[1]) { d[0] = (double)*reinterpret_cast<const short *>(p); }
};
template <> struct Unit<CBGMRES_INT16, 4> {
    static constexpr int EU = 2;
    static __device__ __forceinline__ void load(const unsigned char *p, double (&d)[2]) { i16x2_cvt(*reinterpret_cast<const unsigned *>(p), d[0], d[1]); }
};

struct ConsumerCtx {
    uint64_t *full, *empty, *wfull, *wempty;
    const double *hs_s;
    double *wbuf, *red, *w1buf;
    unsigned char *stages;
    int ns, k, nst; // ring size, columns of this launch, stages per row tile
    int lane, cw, half, ct; // lane, column of the chunk, row half, consumer thread index
};

// One row tile on the consumer side.  acc[ch] are the lane's partial inner products of column
// 8*ch + cw over its rows (kept across tiles); ss / am the lane's partial norms of the new w.
template <int FMT, int F, int KIND, bool RAGGED>
__device__ __forceinline__ void consume_tile(const ConsumerCtx &c, const OrthArgs &a, int64_t r0, int rows, int wslot,
                                             uint32_t wph, Ring &ring, double (&acc)[kMaxChunks], double &ss, double &am)
{
    using T = Tile<FMT, F>;
    constexpr int VEC = T::VEC, GV = T::GV, R = T::R;
    constexpr double PRE = T::Fm::PRE, PRE_EVEN = T::Fm::PRE_EVEN;
    constexpr bool HAS_UPD = KIND != PASS_DOT, HAS_DOT = KIND != PASS_UPD;
    const int wi0 = c.half * T::WORDS_HALF + c.lane; // this lane's first 16-byte word in a column segment
    double *wt = c.wbuf + wslot * R;
    const uint32_t wt_s = smem_u32(wt), red_s = smem_u32(c.red), w1_s = smem_u32(c.w1buf);

    mbar_wait(&c.wfull[wslot], wph);
    if (RAGGED) {
        if constexpr (VEC == 2) { // 1D copy: rows beyond the tile's end read as zero; an odd last row is fetched by hand
            if ((rows & 1) && c.ct == 0) wt[rows - 1] = a.w[r0 + rows - 1];
            for (int r = rows + c.ct; r < R; r += kConsumers) wt[r] = 0.0;
        } else { // 2D box over complete groups of VEC rows (beyond them: zero fill); the last n % VEC rows by hand
            const int64_t nfull = a.n / VEC * VEC;
            if (r0 + rows == a.n && nfull < a.n)
                for (int r = (int)(nfull - r0) + c.ct; r < rows; r += kConsumers) wt[wswz<VEC>(wt_s, r)] = a.w[r0 + r];
            if (nfull == 0) // n < VEC: the map's single group is in range although incomplete
                for (int r = rows + c.ct; r < VEC; r += kConsumers) wt[wswz<VEC>(wt_s, r)] = 0.0;
        }
        consumer_bar();
    }
    // rows of w owned by this lane, pre-multiplied by PRE (see "widening" in device_utils.cuh)
    auto load_w = [&](const double *src, double (&wreg)[GV]) {
        const uint32_t src_s = smem_u32(src);
#pragma unroll
        for (int f = 0; f < F; ++f)
#pragma unroll
            for (int v = 0; v < VEC; v += 2) {
                const double2 t = *reinterpret_cast<const double2 *>(src + wswz<VEC>(src_s, (wi0 + f * 32) * VEC + v));
                wreg[f * VEC + v] = (PRE_EVEN == 1.0) ? t.x : t.x * PRE_EVEN; // even rows: the entries widened by the conversion pipe
                wreg[f * VEC + v + 1] = (PRE == 1.0) ? t.y : t.y * PRE;
            }
    };
    // chunks of stage `st` in which this warp's column exists
    auto valid_chunks = [&](int st) {
        const int left = c.k - st * T::STAGE_COLS - c.cw; // > 0 iff the column exists in chunk 0
        return left <= 0 ? 0 : min(T::CPS, (left + kChunkCols - 1) / kChunkCols);
    };
    // Slots are handed back with mbar_arrive_after_use: `dep` carries a data dependency on everything
    // that was loaded from the slot (device_utils.cuh).
    auto release_w = [&](unsigned dep) {
        if (RAGGED) fence_proxy_async(); // this tile's slot was patched through the generic proxy; the next writer is the TMA
        mbar_arrive_after_use(&c.wempty[wslot], c.lane, dep);
    };
    auto release_stage = [&](int s, unsigned dep) { mbar_arrive_after_use(&c.empty[s], c.lane, dep); };
    auto dep_of = [&](const double(&wreg)[GV]) { // one value per 128-bit load of the w tile
        unsigned dep = 0;
#pragma unroll
        for (int i = 0; i < GV; i += 2) dep ^= dep_bits(wreg[i]);
        return dep;
    };

    if (KIND == PASS_DOT) {
        double wreg[GV];
        load_w(wt, wreg);
#pragma unroll
        for (int st = 0; st < kMaxChunks / T::CPS; ++st) {
            if (st < c.nst) {
                mbar_wait(&c.full[ring.s], ring.ph);
                const unsigned char *stg = c.stages + (size_t)ring.s * T::STAGE;
                for_valid_chunks<FMT, F, RAGGED>(valid_chunks(st), stg, c.cw, wi0, rows, [&](int i, int f, const double(&d)[VEC]) {
                    acc[st * T::CPS + i] += word_dot<VEC>(d, &wreg[f * VEC]);
                });
                unsigned dep = 0;
#pragma unroll
                for (int i = 0; i < T::CPS; ++i) dep ^= dep_bits(acc[st * T::CPS + i]);
                release_stage(ring.s, dep);
                ring.advance(c.ns);
            }
        }
        release_w(dep_of(wreg));
        return;
    }

    const Ring tile_start = ring;
    if constexpr (upd_rowmap<FMT, F, KIND>()) {
        // ---- update, row-owner mapping: this thread's rows, all columns (hs_s holds hs_c unscaled) -----------
        constexpr int UB = 2 * F;
        using U = Unit<FMT, UB>;
        constexpr int EU = U::EU;
        // byte offset of this thread's unit inside a column segment of the stage layout (word_ptr)
        const int ub = c.ct * UB;
        const int uoff = (F == 4) ? (ub >> 11) * T::BOX_BYTES + (ub & 2047) : ub;
        constexpr int CSTR = (F == 4) ? T::BOX_INNER : T::SEG; // distance between columns of a stage
        double pa[EU], pb[EU]; // two chains (even / odd columns)
#pragma unroll
        for (int e = 0; e < EU; ++e) pa[e] = pb[e] = 0.0;
        for (int st = 0; st < c.nst; ++st) {
            const int c0s = st * T::STAGE_COLS;
            const int nc = min(T::STAGE_COLS, c.k - c0s); // columns of this stage that exist (the rest may be stale memory)
            mbar_wait(&c.full[ring.s], ring.ph);
            const unsigned char *base = c.stages + (size_t)ring.s * T::STAGE + uoff;
            int lc = 0;
            for (; lc + 8 <= nc; lc += 8) { // eight columns at a time: all loads first
                double d[8][EU];
                double2 cf[4];
#pragma unroll
                for (int j = 0; j < 8; ++j) U::load(base + (lc + j) * CSTR, d[j]);
#pragma unroll
                for (int j = 0; j < 4; ++j) cf[j] = *reinterpret_cast<const double2 *>(c.hs_s + c0s + lc + 2 * j);
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int e = 0; e < EU; ++e) {
                        pa[e] = fma(d[2 * j][e], cf[j].x, pa[e]);
                        pb[e] = fma(d[2 * j + 1][e], cf[j].y, pb[e]);
                    }
            }
            for (; lc < nc; ++lc) {
                double d[EU];
                U::load(base + lc * CSTR, d);
                const double cf = c.hs_s[c0s + lc];
#pragma unroll
                for (int e = 0; e < EU; ++e) pa[e] = fma(d[e], cf, pa[e]);
            }
            if (KIND == PASS_UPD) release_stage(ring.s, dep_bits(pa[0]) ^ dep_bits(pb[0]));
            ring.advance(c.ns);
        }
        // new w of this thread's rows.  Two buffers for the second sweep, alternating by tile: no barrier
        // separates a fast thread's writes for this tile from a slow thread's reads of the previous one
        // (the unused `red` area is the second buffer).
        double *w1 = (wslot & 1) ? c.red : c.w1buf;
        const uint32_t w1r_s = smem_u32(w1);
        const int rbase = c.ct * EU;
        double wn[EU];
#pragma unroll
        for (int e = 0; e < EU; ++e) {
            const int r = rbase + e;
            wn[e] = wt[wswz<VEC>(wt_s, r)] - (pa[e] + pb[e]);
            const bool live = !RAGGED || r < rows;
            if (live) {
                ss = fma(wn[e], wn[e], ss);
                am = fmax(am, fabs(wn[e]));
            } else wn[e] = 0.0;
            if (HAS_DOT) w1[wswz<VEC>(w1r_s, r)] = wn[e]; // kept apart from the TMA-written slot: no proxy fence
        }
        if (EU == 2 && (!RAGGED || rbase + 1 < rows)) *reinterpret_cast<double2 *>(a.w + r0 + rbase) = make_double2(wn[0], wn[EU - 1]);
        else {
#pragma unroll
            for (int e = 0; e < EU; ++e)
                if (!RAGGED || rbase + e < rows) a.w[r0 + rbase + e] = wn[e];
        }
        if (HAS_DOT) consumer_bar(); // every row of w1buf is in place before the second sweep reads it
        release_w(dep_bits(wn[0]));
        if (KIND == PASS_UPD) return;
    } else {
    // ---- update: p = sum_c dec(V)[rows, c] * hs_c over this warp's columns (hs_s holds PRE * hs_c) ------
    double p[GV];
#pragma unroll
    for (int i = 0; i < GV; ++i) p[i] = 0.0;
    for (int st = 0; st < c.nst; ++st) {
        double coef[T::CPS], coefE[T::CPS]; // zero beyond k; coefE: for the even entries (mixed widening)
#pragma unroll
        for (int i = 0; i < T::CPS; ++i) {
            coef[i] = c.hs_s[st * T::STAGE_COLS + i * kChunkCols + c.cw];
            coefE[i] = (PRE_EVEN == PRE) ? coef[i] : coef[i] * (PRE_EVEN / PRE);
        }
        mbar_wait(&c.full[ring.s], ring.ph);
        const unsigned char *stg = c.stages + (size_t)ring.s * T::STAGE;
        for_valid_chunks<FMT, F, RAGGED>(valid_chunks(st), stg, c.cw, wi0, rows, [&](int i, int f, const double(&d)[VEC]) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) p[f * VEC + v] = fma(d[v], (v & 1) ? coef[i] : coefE[i], p[f * VEC + v]);
        });
        if (KIND == PASS_UPD) {
            unsigned dep = 0; // p[f * VEC] has consumed word f of every column of the stage
#pragma unroll
            for (int f = 0; f < F; ++f) dep ^= dep_bits(p[f * VEC]);
            release_stage(ring.s, dep);
        }
        ring.advance(c.ns);
    }
    double *redw = c.red + c.cw * R;
    const uint32_t redw_s = smem_u32(redw);
#pragma unroll
    for (int f = 0; f < F; ++f)
#pragma unroll
        for (int v = 0; v < VEC; v += 2)
            *reinterpret_cast<double2 *>(redw + wswz<VEC>(redw_s, (wi0 + f * 32) * VEC + v)) = make_double2(p[f * VEC + v], p[f * VEC + v + 1]);
    half_bar(c.half);
    // new w of this half's rows: the eight partial row vectors are added in a fixed order
    for (int r = c.half * (R / 2) + (c.ct & (kConsumers / 2 - 1)); r < (c.half + 1) * (R / 2); r += kConsumers / 2) {
        double tot = 0.0;
#pragma unroll
        for (int q = 0; q < kColWarps; ++q) tot += c.red[q * R + wswz<VEC>(red_s + q * R * 8, r)]; // stored like the w tiles: conflict-free both ways
        const double wo = wt[wswz<VEC>(wt_s, r)];
        const double wn = (PRE == 1.0) ? wo - tot : fma(-tot, PRE, wo); // tot * PRE is exact: one rounding either way
        const bool live = !RAGGED || r < rows;
        if (live) {
            a.w[r0 + r] = wn;
            ss = fma(wn, wn, ss);
            am = fmax(am, fabs(wn));
        }
        if (HAS_DOT) c.w1buf[wswz<VEC>(w1_s, r)] = live ? wn : 0.0; // kept apart from the TMA-written slot: no proxy fence
    }
    half_bar(c.half);
    release_w(dep_bits(ss)); // the tile of w was consumed by the stores of the new w and by the norms
    if (KIND == PASS_UPD) return;
    }

    // ---- second sweep over the resident chunks: u_c += sum_rows dec(V)[r, c] * w_new[r] -----------------
    double wreg[GV];
    load_w((upd_rowmap<FMT, F, KIND>() && (wslot & 1)) ? c.red : c.w1buf, wreg);
    Ring r2 = tile_start;
#pragma unroll
    for (int st = 0; st < kMaxChunks / T::CPS; ++st) {
        if (st < c.nst) {
            const unsigned char *stg = c.stages + (size_t)r2.s * T::STAGE;
            for_valid_chunks<FMT, F, RAGGED>(valid_chunks(st), stg, c.cw, wi0, rows, [&](int i, int f, const double(&d)[VEC]) {
                acc[st * T::CPS + i] += word_dot<VEC>(d, &wreg[f * VEC]);
            });
            unsigned dep = 0;
#pragma unroll
            for (int i = 0; i < T::CPS; ++i) dep ^= dep_bits(acc[st * T::CPS + i]);
            release_stage(r2.s, dep);
            r2.advance(c.ns);
        }
    }
    (void)HAS_UPD;
}


// ---- final stage, run by the CTA that finished last ---------------------------------------------------
// Adds the CTA partials in a fixed order, applies the per-vector scales (h_c = sigma_c * sum q w),
// and takes the decisions of Fig. 1 l.6-12 from the norms of the new w.
template <int KIND, bool SCALED> __device__ void orth_finalize(const OrthArgs &a, int k, double *scratch)
{
    constexpr bool HAS_UPD = KIND != PASS_DOT, HAS_DOT = KIND != PASS_UPD;
    constexpr int NW = kOrthThreads / 32;
    constexpr int UNR = 19; // partials in flight per thread: the loads are L2 round trips, issue them together
    Ctl *ctl = a.ctl;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nb = gridDim.x;
    __shared__ int s_apply;
    __shared__ double s_nrm[2 * NW];
    if (tid == 0) s_apply = 1;

    // ---- loads first: every thread's share of the CTA partials, all in flight at once ----------------
    double nt = 0.0, nm = 0.0; // norms: one CTA per thread (grid <= kOrthThreads)
    if (HAS_UPD && a.last_range && tid < nb) {
        nt = __ldcg(&a.npart[tid]);
        nm = __ldcg(&a.npart[kMaxGrid + tid]);
    }
    // dots: columns padded to kc = 32, 64 or 128; 512 / kc slices of CTAs, slice sl adds CTAs
    // [sl * per, (sl + 1) * per) of its column in a fixed order
    const int kc = k <= 32 ? 32 : (k <= 64 ? 64 : 128);
    const int nsl = 512 / kc, col = tid & (kc - 1), sl = tid / kc;
    const int per = (nb + nsl - 1) / nsl;
    double *part = scratch; // [nsl][kMaxRangeCols]
    // sigma_c of the column this thread finishes below: fetched with the partials, not after them
    double sigma_v = 1.0;
    if (HAS_DOT && SCALED && tid < k) sigma_v = __ldcg(&a.scales[tid]);
    if (HAS_DOT && tid < 512) {
        double sum = 0.0;
        if (col < k) {
            const int b1 = min(nb, (sl + 1) * per);
            for (int b = sl * per; b < b1; b += UNR) {
                double v[UNR];
#pragma unroll
                for (int u = 0; u < UNR; ++u) v[u] = (b + u < b1) ? __ldcg(&a.partials[(size_t)(b + u) * kLdp + col]) : 0.0;
#pragma unroll
                for (int u = 0; u < UNR; ++u) sum += v[u];
            }
        }
        part[sl * kMaxRangeCols + col] = sum;
    }
    if (HAS_UPD && a.last_range) {
        nt = warp_sum(nt);
        nm = warp_max(nm);
        if (lane == 0) {
            s_nrm[warp] = nt;
            s_nrm[NW + warp] = nm;
        }
    }
    __syncthreads();
    if (HAS_UPD && a.last_range && tid == 0) {
        double t = 0.0, m = 0.0;
#pragma unroll
        for (int i = 0; i < NW; ++i) {
            t += s_nrm[i];
            m = fmax(m, s_nrm[NW + i]);
        }
        const double hn = sqrt(t);
        if (a.mode == MODE_HOOK) {
            ctl->hook_nrm2 = hn;
            ctl->hook_amax = m;
        } else if (a.mode == MODE_ORTH1) {
            // Fig. 1 l.6-7: h_{j+1,j} := ||w||_2 ; re-orthogonalise iff h_{j+1,j} < eta * omega
            const int flag = (ctl->reorth_mode == CBGMRES_REORTH_ALWAYS) ||
                             (ctl->reorth_mode == CBGMRES_REORTH_COND && hn < ctl->eta * ctl->omega);
            ctl->hn = hn;
            ctl->amax = m;
            ctl->breakdown = (hn == 0.0);
            ctl->reorth_flag = flag;
            ctl->reorth_log[a.step] = (unsigned char)flag;
            if (!isfinite(hn)) ctl->nonfinite = 1;
            s_apply = flag;
        } else if (a.mode == MODE_ORTH2) {
            // Fig. 1 l.10-12: new norm; breakdown if it again fell below eta * (norm before the pass)
            const double omega1 = ctl->hn;
            ctl->hn = hn;
            ctl->amax = m;
            ctl->reorth_count += 1;
            ctl->breakdown = (hn == 0.0) || (hn < ctl->eta * omega1);
            if (!isfinite(hn)) ctl->nonfinite = 1;
        }
    }
    if (HAS_UPD && HAS_DOT) __syncthreads(); // s_apply
    if (HAS_DOT) {
        const bool apply = s_apply != 0;
        for (int c = tid; c < k; c += kOrthThreads) { // k <= kMaxRangeCols < kOrthThreads: c == tid
            double tot = 0.0;
            for (int q = 0; q < nsl; ++q) tot += part[q * kMaxRangeCols + c];
            const double sigma = sigma_v;
            const double h = tot * sigma; // h_c = sigma_c * sum_i q_ic w_i
            if (KIND == PASS_DOT) {
                if (a.mode == MODE_ORTH2) a.h_out[c] += h; // Fig. 1 l.9: h_{1:j,j} += u
                else a.h_out[c] = h;
                if (a.hs_out) a.hs_out[c] = h * sigma;     // coefficient of the raw payload in the update
            } else if (a.mode == MODE_HOOK) {
                a.h_out[c] = h;
                if (a.hs_out) a.hs_out[c] = h * sigma;
            } else if (apply) { // fused pass inside the solver: u only counts if the second pass fires (l.7-9)
                a.h_out[c] += h;
                a.hs_out[c] = h * sigma;
            }
        }
    }
    if (a.mode != MODE_HOOK && a.last_range && tid == 0) ctl->dir ^= 1;
}

template <int FMT, int F, int KIND>
__global__ void __launch_bounds__(kOrthThreads, 1)
    orth_kernel(const OrthArgs a, const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap wmap)
{
    using T = Tile<FMT, F>;
    constexpr int R = T::R, B = T::B;
    constexpr bool HAS_UPD = KIND != PASS_DOT, HAS_DOT = KIND != PASS_UPD;
    Ctl *ctl = a.ctl;
    const int ns = a.nstages;

    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    uint64_t *empty = full + kMaxStages;
    uint64_t *wfull = empty + kMaxStages;
    uint64_t *wempty = wfull + kWSlots;
    double *hs_s = reinterpret_cast<double *>(smem + 1024);
    double *hpart = reinterpret_cast<double *>(smem + 2048);
    double *wbuf = reinterpret_cast<double *>(smem + 4096);
    double *red = wbuf + kWSlots * R;
    unsigned char *stages = smem + orth_fixed_smem(R, HAS_UPD);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < ns; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kConsumerWarps);
        }
        for (int s = 0; s < kWSlots; ++s) {
            mbar_init(&wfull[s], 1);
            mbar_init(&wempty[s], kConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // Row tiles of this CTA.  Interleaved (default): tile t belongs to CTA t mod grid, so the CTAs
    // sweep a contiguous window of the basis together.  Blocked: one contiguous row range per CTA (a
    // multiple of 64 rows, so every tile start is 16-byte aligned in every format).
    int64_t row_begin, row_end, tile_stride;
    int ntiles;
    if (a.interleave) {
        const int64_t total = (a.n + R - 1) / R;
        ntiles = (int)((total - blockIdx.x + gridDim.x - 1) / gridDim.x);
        if (ntiles < 0) ntiles = 0;
        row_begin = (int64_t)blockIdx.x * R;
        row_end = a.n;
        tile_stride = (int64_t)gridDim.x * R;
    } else {
        const int64_t per = ((a.n + gridDim.x - 1) / gridDim.x + 63) / 64 * 64;
        row_begin = min(a.n, (int64_t)blockIdx.x * per);
        row_end = min(a.n, row_begin + per);
        ntiles = (int)((row_end - row_begin + R - 1) / R);
        tile_stride = R;
    }
    const int dir = a.dir; // consecutive passes of a step walk in opposite directions (set by the host)

    // One stage of row tile (first row r0) into ring slot `slot`: lane 0 arms the barrier, lanes 0..3 issue the boxes.
    auto issue_stage = [&](int64_t r0, int st, int slot, int kk) {
        const int x0 = (int)(r0 * B / 8); // first 8-byte word of the tile inside a column
        const int c_first = st * T::STAGE_COLS;
        // boxes of this stage that hold at least one wanted column (F = 4: both halves of 8 columns)
        const int nboxes = (F == 4) ? T::BOXES : min(T::BOXES, (kk - c_first + kChunkCols - 1) / kChunkCols);
        if (lane == 0) mbar_expect_tx(&full[slot], nboxes * T::BOX_BYTES);
        __syncwarp();
        if (lane < nboxes) {
            unsigned char *dst = stages + (size_t)slot * T::STAGE + lane * T::BOX_BYTES;
            if (F == 4) tma_box_g2s(dst, &tmap, x0 + lane * (T::BOX_INNER / 8), c_first, &full[slot]);
            else tma_box_g2s(dst, &tmap, x0, c_first + lane * kChunkCols, &full[slot]);
        }
    };

    // ---- before the grid dependency resolves: the basis is not written by the predecessor kernel (the
    // store of the newest vector completed before the predecessor started), so the producer already
    // fetches the first stages of the first row tile while the predecessor's tail -- its last CTAs and
    // the last-block-done final stage -- is still running.  Nothing else is read before the wait.
    int pre = 0;
    if (warp == kConsumerWarps && !a.d_k && ntiles > 0) {
        const int nst0 = (a.k + T::STAGE_COLS - 1) / T::STAGE_COLS;
        pre = nst0 < ns ? nst0 : ns;
        const int t0 = dir ? ntiles - 1 : 0;
        for (int st = 0; st < pre; ++st) issue_stage(row_begin + (int64_t)t0 * tile_stride, st, st, a.k);
    }
    pdl_wait();
    pdl_launch_dependents();
    // the control words this CTA needs, fetched together (each is an L2 round trip)
    const int stop_after = __ldcg(&ctl->stop_after), reorth_flag = __ldcg(&ctl->reorth_flag);
    const int dk = a.d_k ? __ldcg(a.d_k) : 0;
    double hs_v = 0.0; // this thread's update coefficient, fetched in the same round trip as the control words
    if (HAS_UPD && tid < a.k) hs_v = __ldcg(&a.hs[tid]);
    int k = a.k;
    bool run = true;
    if (a.mode == MODE_ORTH1 || a.mode == MODE_ORTH2) {
        if (a.step > stop_after) run = false;
        if (a.mode == MODE_ORTH2 && !reorth_flag) run = false;
    }
    if (a.d_k) { // cycle-end x update: the number of basis vectors is only known on the device
        k = min(a.k, dk - a.c0);
        if (k <= 0) run = false;
    }
    if (!run) { // copies in flight must land before the CTA gives its shared memory back
        if (warp == kConsumerWarps && lane == 0)
            for (int s = 0; s < pre; ++s) mbar_wait(&full[s], 0u);
        return;
    }
    const int nst = (k + T::STAGE_COLS - 1) / T::STAGE_COLS; // stages per row tile
    if (HAS_UPD && tid < kConsumers) {
        if (tid < kMaxRangeCols) hs_s[tid] = (tid < k) ? hs_v * (upd_rowmap<FMT, F, KIND>() ? 1.0 : T::Fm::PRE) : 0.0;
        consumer_bar();
    }

    double acc[kMaxChunks];
#pragma unroll
    for (int i = 0; i < kMaxChunks; ++i) acc[i] = 0.0;
    double ss = 0.0, am = 0.0;

    if (warp == kConsumerWarps) {
        // ---- producer: one elected lane waits for free slots, lanes 0..7 issue one column copy each ----
        Ring ring;
        for (int i = 0; i < ntiles; ++i) {
            const int t = dir ? ntiles - 1 - i : i;
            const int64_t r0 = row_begin + (int64_t)t * tile_stride;
            const int rows = (int)min((int64_t)R, row_end - r0);
            const uint32_t w_bytes = (T::VEC == 2) ? ((uint32_t)(rows * 8) & ~15u) : (uint32_t)(R * 8);
            const int wslot = i % kWSlots;
            if (lane == 0) {
                mbar_wait(&wempty[wslot], ((i / kWSlots) & 1) ^ 1u);
                mbar_expect_tx(&wfull[wslot], w_bytes);
                if constexpr (T::VEC == 2) { // linear tile, 1D bulk copy
                    if (w_bytes) bulk_g2s(wbuf + wslot * R, a.w + r0, w_bytes, &wfull[wslot]);
                } else { // swizzled tile: box [VEC x R / VEC] of w seen as [n / VEC][VEC]
                    tma_box_g2s(wbuf + wslot * R, &wmap, 0, (int)(r0 / T::VEC), &wfull[wslot]);
                }
            }
            for (int st = 0; st < nst; ++st) {
                if (i > 0 || st >= pre) { // (the first `pre` stages of the first tile are already on their way)
                    if (lane == 0) mbar_wait(&empty[ring.s], ring.ph ^ 1u);
                    issue_stage(r0, st, ring.s, k);
                }
                ring.advance(ns);
            }
        }
    } else {
        ConsumerCtx c{full, empty, wfull, wempty, hs_s, wbuf, red, red + kColWarps * R, stages, ns, k, nst, lane, warp & 7, warp >> 3, tid};
        Ring ring;
        for (int i = 0; i < ntiles; ++i) {
            const int t = dir ? ntiles - 1 - i : i;
            const int64_t r0 = row_begin + (int64_t)t * tile_stride;
            const int rows = (int)min((int64_t)R, row_end - r0);
            if (rows == R) consume_tile<FMT, F, KIND, false>(c, a, r0, rows, i % kWSlots, (i / kWSlots) & 1, ring, acc, ss, am);
            else consume_tile<FMT, F, KIND, true>(c, a, r0, rows, i % kWSlots, (i / kWSlots) & 1, ring, acc, ss, am);
        }
        // ---- CTA partials ------------------------------------------------------------------------------
        if (HAS_DOT) {
            const double tot = butterfly_rec<kMaxChunks, 16>(acc, lane);
            if (butterfly_owner<kMaxChunks>(lane)) {
                const int col = butterfly_col<kMaxChunks>(lane) * kChunkCols + (warp & 7);
                hpart[(warp >> 3) * kMaxRangeCols + col] = tot * T::Fm::PRE; // acc holds sums / PRE
            }
        }
        if (HAS_UPD) {
            ss = warp_sum(ss);
            am = warp_max(am);
            consumer_bar(); // the other row half may still be adding the partial row vectors of its last tile out of `red`
            if (lane == 0) {
                red[warp] = ss;
                red[kConsumerWarps + warp] = am;
            }
        }
    }
    __syncthreads();
    if (HAS_DOT)
        for (int col = tid; col < k; col += kOrthThreads)
            a.partials[(size_t)blockIdx.x * kLdp + col] = hpart[col] + hpart[kMaxRangeCols + col];
    if (HAS_UPD && tid == 0) {
        double t = 0.0, m = 0.0;
        for (int i = 0; i < kConsumerWarps; ++i) {
            t += red[i];
            m = fmax(m, red[kConsumerWarps + i]);
        }
        a.npart[blockIdx.x] = t;
        a.npart[kMaxGrid + blockIdx.x] = m;
    }
    if (!last_block_done(&ctl->tickets[0])) return;
    orth_finalize<KIND, T::Fm::SCALED>(a, k, reinterpret_cast<double *>(smem + 4096));
}


// ---- fused update + multi-dot for the reduced formats: warps own rows, lane groups own columns ---------------
// The column-mapped fused kind above pays a k-INDEPENDENT price per row: the eight partial row vectors of a
// tile go through shared memory (160 bytes of shared-memory traffic per row) between two CTA-wide barriers
// that put all sixteen warps in lock-step -- measured (clock64 probes, n = 4.2e6, fp16): 40 % of a tile's time
// is barrier / data wait, and the pass costs ~57 us more than its bytes at every k.  Here the 32 lanes of a
// warp are 8 groups of 4: group j owns column 8 ch + j of every 8-column chunk, its four lanes own the 16-byte
// payload words of the warp's rows (64 or 128 bytes of each column segment per warp).  The partial sums of
// the update are then spread over the lane GROUPS of one warp and are added by a transposing butterfly of
// shuffles -- no shared memory, no barrier, the sixteen warps drift apart and hide each other's latencies.
// The new w leaves the lane that holds the finished row (global store + a per-warp shared buffer for the
// second sweep, __syncwarp only); w itself is fetched from global memory into registers at the start of the
// tile, so there is no w ring either.
// Shared-memory layout of a chunk: the basis is seen as the 3D array [128-byte segments][columns][16 words]
// and a TMA box [16 words x 8 columns x SEGS segments] lands as rows rho = 8 seg + col of 128 bytes with the
// 128-byte swizzle (16-byte chunk index XOR rho mod 8 = col): the four lanes of each of the eight groups hit
// all eight 16-byte bank groups four times per 512-byte wavefront set -- the minimum for a 128-bit warp load.
constexpr int kFGroups = 8; // lane groups per warp = columns per chunk

template <int FMT, int WPL> struct FTile {
    using Fm = Fmt<FMT>;
    static constexpr int VEC = Fm::VEC, B = Fm::BYTES;
    static constexpr int SEGS = 8 * WPL;                 // 128-byte segments per column segment
    static constexpr int SEG = SEGS * 128;               // 1 or 2 KB per column and tile
    static constexpr int R = SEG / B;                    // rows of a tile
    static constexpr int RW = R / kConsumerWarps;        // rows of a warp (64 * WPL bytes of every column)
    static constexpr int NV = VEC * WPL;                 // rows of a lane
    static constexpr int BOX_BYTES = kFGroups * SEG;     // one chunk of 8 columns: 8 or 16 KB
    static constexpr int CPS = kStageBytes / BOX_BYTES;  // chunks per 32 KB stage: 4 or 2
    static constexpr int STAGE_COLS = CPS * kFGroups;
    static constexpr int W1_BYTES = R * 8;               // the new w of the tile, per-warp slices
};
__host__ __device__ constexpr int ffixed_smem(int R) { return 2048 + R * 8; } // barriers, coefficients, w1 (then 1 KB-aligned stages)

__device__ __forceinline__ void tma_box3_g2s(void *dst_smem, const CUtensorMap *map, int x, int y, int z, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dst_smem)),
        "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
        : "memory");
}

// Transposing butterfly over the 8 lane groups (lane bits 4, 3, 2): every lane holds N partial sums (one per row
// of its payload words, summed over the columns of ITS group); afterwards the lane holds max(1, N / 8) finished
// sums, those with index fgroup_first<N>(lane) ... (for N < 8 both lanes of a pair hold the same sum).
template <int N, int OFF, int NOUT> __device__ __forceinline__ void fgroup_reduce(double (&a)[N], int lane, double (&out)[NOUT])
{
    if constexpr (OFF < 4) {
        static_assert(N == NOUT, "butterfly ends with NOUT sums per lane");
#pragma unroll
        for (int i = 0; i < N; ++i) out[i] = a[i];
    } else if constexpr (N == 1) {
        double b[1] = {a[0] + shfl_xor_f64(a[0], OFF)};
        fgroup_reduce<1, OFF / 2, NOUT>(b, lane, out);
    } else {
        constexpr int H = N / 2;
        const bool up = (lane & OFF) != 0;
        double b[H];
#pragma unroll
        for (int i = 0; i < H; ++i) {
            const double send = up ? a[i] : a[i + H];
            const double keep = up ? a[i + H] : a[i];
            b[i] = keep + shfl_xor_f64(send, OFF);
        }
        fgroup_reduce<H, OFF / 2, NOUT>(b, lane, out);
    }
}
// index (into the lane's N rows) of the first finished sum a lane holds after fgroup_reduce<N, 16>
template <int N> __device__ __forceinline__ int fgroup_first(int lane)
{
    int idx = 0, n = N;
#pragma unroll
    for (int off = 16; off >= 4; off >>= 1) {
        if (n > 1) {
            n >>= 1;
            if (lane & off) idx += n;
        }
    }
    return idx;
}

template <int FMT, int WPL>
__global__ void __launch_bounds__(kOrthThreads, 1)
    orth_fused_kernel(const OrthArgs a, const __grid_constant__ CUtensorMap tmap)
{
    using T = FTile<FMT, WPL>;
    using Fm = typename T::Fm;
    constexpr int VEC = T::VEC, B = T::B, R = T::R, NV = T::NV, RW = T::RW;
    constexpr int NOUT = NV >= 8 ? NV / 8 : 1; // finished rows per lane after the butterfly
    constexpr double PRE = Fm::PRE, PRE_EVEN = Fm::PRE_EVEN;
    Ctl *ctl = a.ctl;
    const int ns = a.nstages;

    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u); // the swizzle pattern repeats every 1 KB
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    uint64_t *empty = full + kMaxStages;
    double *hs_s = reinterpret_cast<double *>(smem + 1024);
    double *w1 = reinterpret_cast<double *>(smem + 2048);
    unsigned char *stages = smem + ((ffixed_smem(R) + 1023) & ~1023);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < ns; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // row tiles dealt round-robin to the CTAs (the CTAs sweep a contiguous window of the basis together)
    const int64_t total = (a.n + R - 1) / R;
    int ntiles = (int)((total - blockIdx.x + gridDim.x - 1) / gridDim.x);
    if (ntiles < 0) ntiles = 0;
    const int64_t row_begin = (int64_t)blockIdx.x * R, tile_stride = (int64_t)gridDim.x * R;
    const int dir = a.dir;

    auto issue_stage = [&](int64_t r0, int st, int slot, int kk) { // lanes 0..CPS-1 issue one chunk each
        const int c_first = st * T::STAGE_COLS;
        const int nboxes = min(T::CPS, (kk - c_first + kFGroups - 1) / kFGroups);
        if (lane == 0) mbar_expect_tx(&full[slot], nboxes * T::BOX_BYTES);
        __syncwarp();
        if (lane < nboxes)
            tma_box3_g2s(stages + (size_t)slot * kStageBytes + lane * T::BOX_BYTES, &tmap, 0, c_first + lane * kFGroups,
                         (int)(r0 * B / 128), &full[slot]);
    };

    // the basis is not written by the predecessor kernel: first stages before the grid dependency resolves
    int pre = 0;
    if (warp == kConsumerWarps && ntiles > 0) {
        const int nst0 = (a.k + T::STAGE_COLS - 1) / T::STAGE_COLS;
        pre = nst0 < ns ? nst0 : ns;
        const int t0 = dir ? ntiles - 1 : 0;
        for (int st = 0; st < pre; ++st) issue_stage(row_begin + (int64_t)t0 * tile_stride, st, st, a.k);
    }
    pdl_wait();
    pdl_launch_dependents();
    const int stop_after = __ldcg(&ctl->stop_after);
    double hs_v = 0.0;
    if (tid < a.k) hs_v = __ldcg(&a.hs[tid]);
    const int k = a.k;
    if (a.mode == MODE_ORTH1 && a.step > stop_after) { // copies in flight must land before the CTA gives its shared memory back
        if (warp == kConsumerWarps && lane == 0)
            for (int s = 0; s < pre; ++s) mbar_wait(&full[s], 0u);
        return;
    }
    const int nst = (k + T::STAGE_COLS - 1) / T::STAGE_COLS;
    if (tid < kConsumers) {
        if (tid < kMaxRangeCols) hs_s[tid] = (tid < k) ? hs_v * PRE : 0.0;
        consumer_bar();
    }

    double acc[kMaxChunks];
#pragma unroll
    for (int i = 0; i < kMaxChunks; ++i) acc[i] = 0.0;
    double ss = 0.0, am = 0.0;

    if (warp == kConsumerWarps) {
        // ---- producer --------------------------------------------------------------------------------------
        Ring ring;
        for (int i = 0; i < ntiles; ++i) {
            const int t = dir ? ntiles - 1 - i : i;
            const int64_t r0 = row_begin + (int64_t)t * tile_stride;
            for (int st = 0; st < nst; ++st) {
                if (i > 0 || st >= pre) {
                    if (lane == 0) mbar_wait(&empty[ring.s], ring.ph ^ 1u);
                    issue_stage(r0, st, ring.s, k);
                }
                ring.advance(ns);
            }
        }
    } else {
        // ---- consumers: warp w owns rows [w RW, (w+1) RW) of every tile; lane = (group j, word t) -----------
        const int j = lane >> 2, t4 = lane & 3;
        // byte offset of this lane's word(s) inside a chunk: row rho = 8 seg + j of 128 bytes, 16-byte chunk c ^ j
        int woff[WPL], rloc[WPL]; // ... and the first row (within the warp's rows) each word covers
        if constexpr (WPL == 1) {
            const int seg = warp >> 1, c = 4 * (warp & 1) + t4;
            woff[0] = (seg * 8 + j) * 128 + ((c ^ j) & 7) * 16;
            rloc[0] = t4 * VEC;
        } else {
#pragma unroll
            for (int q = 0; q < WPL; ++q) {
                const int c = t4 + 4 * q;
                woff[q] = (warp * 8 + j) * 128 + ((c ^ j) & 7) * 16;
                rloc[q] = c * VEC;
            }
        }
        double *w1w = w1 + warp * RW; // this warp's slice of the new w
        const int ofirst = fgroup_first<NV>(lane); // index among the lane's NV rows of the row(s) it finishes
        // rows (within the warp) this lane finishes: NV rows are ordered word 0 rows, word 1 rows
        const int fin_r = rloc[ofirst / VEC] + (ofirst % VEC);
        const bool fin_owner = NV >= 8 || (lane & (NV == 4 ? 4 : 12)) == 0; // for N < 8 several lanes hold the same sum: one writes
        Ring ring;
        for (int i = 0; i < ntiles; ++i) {
            const int t = dir ? ntiles - 1 - i : i;
            const int64_t r0 = row_begin + (int64_t)t * tile_stride;
            const int64_t rows_left = a.n - r0; // rows of the tile that exist (may exceed R)
            // the tile body, compiled twice: RAGGED = the tile runs past row n (masks per entry), else no masks
            auto tile = [&](auto ragged_tag) {
            constexpr bool ragged = decltype(ragged_tag)::value;
            const int64_t gr = r0 + warp * RW + fin_r; // global row of the first row this lane finishes
            // old w of the rows this lane will finish: in flight during the first sweep
            double wold[NOUT];
#pragma unroll
            for (int e = 0; e < NOUT; ++e) wold[e] = 0.0;
            if (fin_owner) {
                if (NOUT == 2 && gr + 1 < a.n) {
                    const double2 v2 = __ldcg(reinterpret_cast<const double2 *>(a.w + gr));
                    wold[0] = v2.x;
                    wold[NOUT - 1] = v2.y;
                } else {
#pragma unroll
                    for (int e = 0; e < NOUT; ++e)
                        if (gr + e < a.n) wold[e] = __ldcg(a.w + gr + e);
                }
            }
            // rows of this lane's words that exist (ragged tile): word q covers warp rows rloc[q] .. rloc[q] + VEC
            int live[WPL];
#pragma unroll
            for (int q = 0; q < WPL; ++q) {
                const int64_t left = rows_left - (warp * RW + rloc[q]);
                live[q] = ragged ? (int)max((int64_t)0, min((int64_t)VEC, left)) : VEC;
            }
            const Ring tile_start = ring;
            // ---- sweep 1: p = sum over this group's columns of dec(V)[rows, c] * hs_c ---------------------------
            double p[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) p[v] = 0.0;
            for (int st = 0; st < nst; ++st) {
                mbar_wait(&full[ring.s], ring.ph);
                const unsigned char *stg = stages + (size_t)ring.s * kStageBytes;
                const int nch = min(T::CPS, (k - st * T::STAGE_COLS + kFGroups - 1) / kFGroups); // chunks with a wanted column
                // NC = chunks of this stage that hold a wanted column (CPS for every stage but a tile's last):
                // all loads first, then the NC * WPL independent decode + FMA chains
                auto chunks = [&](auto nc_tag) {
                    constexpr int NC = decltype(nc_tag)::value;
                    uint4 raw[NC][WPL];
                    double coef[NC], coefE[NC]; // coefE: for the even entries (mixed widening)
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        coef[c] = hs_s[st * T::STAGE_COLS + c * kFGroups + j]; // zero beyond k
                        coefE[c] = (PRE_EVEN == PRE) ? coef[c] : coef[c] * (PRE_EVEN / PRE);
#pragma unroll
                        for (int q = 0; q < WPL; ++q)
                            raw[c][q] = (live[q] > 0) ? *reinterpret_cast<const uint4 *>(stg + c * T::BOX_BYTES + woff[q])
                                                      : make_uint4(0u, 0u, 0u, 0u);
                    }
#pragma unroll
                    for (int c = 0; c < NC; ++c)
#pragma unroll
                        for (int q = 0; q < WPL; ++q) {
                            double d[VEC];
                            Fm::decode(raw[c][q], d);
#pragma unroll
                            for (int v = 0; v < VEC; ++v) {
                                if (ragged && v >= live[q]) d[v] = 0.0; // padding beyond n may decode to anything
                                p[q * VEC + v] = fma(d[v], (v & 1) ? coef[c] : coefE[c], p[q * VEC + v]);
                            }
                        }
                };
                if (nch >= T::CPS) chunks(std::integral_constant<int, T::CPS>{});
                else if (nch == 1) chunks(std::integral_constant<int, 1>{});
                else if constexpr (T::CPS == 4) {
                    if (nch == 2) chunks(std::integral_constant<int, 2>{});
                    else chunks(std::integral_constant<int, 3>{});
                }
                ring.advance(ns);
            }
            // ---- the partial sums of the 8 groups -> finished rows; new w ---------------------------------------
            double tot[NOUT];
            fgroup_reduce<NV, 16, NOUT>(p, lane, tot);
            double wn[NOUT];
#pragma unroll
            for (int e = 0; e < NOUT; ++e) {
                wn[e] = (PRE == 1.0) ? wold[e] - tot[e] : fma(-tot[e], PRE, wold[e]); // tot * PRE is exact: one rounding either way
                const bool exists = gr + e < a.n;
                if (!exists) wn[e] = 0.0;
                if (fin_owner && exists) {
                    ss = fma(wn[e], wn[e], ss);
                    am = fmax(am, fabs(wn[e]));
                }
            }
            if (fin_owner) {
                if (NOUT == 2) {
                    *reinterpret_cast<double2 *>(w1w + fin_r) = make_double2(wn[0], wn[NOUT - 1]);
                    if (gr + 1 < a.n) *reinterpret_cast<double2 *>(a.w + gr) = make_double2(wn[0], wn[NOUT - 1]);
                    else if (gr < a.n) a.w[gr] = wn[0];
                } else {
                    w1w[fin_r] = wn[0];
                    if (gr < a.n) a.w[gr] = wn[0];
                }
            }
            __syncwarp();
            // ---- sweep 2 over the resident chunks: u_c += sum_rows dec(V)[r, c] * w_new[r] ----------------------
            double wreg[NV];
#pragma unroll
            for (int q = 0; q < WPL; ++q)
#pragma unroll
                for (int v = 0; v < VEC; v += 2) {
                    const double2 t2 = *reinterpret_cast<const double2 *>(w1w + rloc[q] + v);
                    wreg[q * VEC + v] = (PRE_EVEN == 1.0) ? t2.x : t2.x * PRE_EVEN;
                    wreg[q * VEC + v + 1] = (PRE == 1.0) ? t2.y : t2.y * PRE;
                }
            __syncwarp(); // w1w is rewritten by the next tile only after every lane has read it
            Ring r2 = tile_start;
#pragma unroll
            for (int st = 0; st < kMaxChunks / T::CPS; ++st) {
                if (st < nst) {
                    const unsigned char *stg = stages + (size_t)r2.s * kStageBytes;
                    const int nch = min(T::CPS, (k - st * T::STAGE_COLS + kFGroups - 1) / kFGroups);
                    auto chunks = [&](auto nc_tag) {
                        constexpr int NC = decltype(nc_tag)::value;
                        uint4 raw[NC][WPL];
#pragma unroll
                        for (int c = 0; c < NC; ++c)
#pragma unroll
                            for (int q = 0; q < WPL; ++q)
                                raw[c][q] = (live[q] > 0) ? *reinterpret_cast<const uint4 *>(stg + c * T::BOX_BYTES + woff[q])
                                                          : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
                        for (int c = 0; c < NC; ++c)
#pragma unroll
                            for (int q = 0; q < WPL; ++q) {
                                double d[VEC];
                                Fm::decode(raw[c][q], d);
                                if (ragged) {
#pragma unroll
                                    for (int v = 0; v < VEC; ++v)
                                        if (v >= live[q]) d[v] = 0.0;
                                }
                                acc[st * T::CPS + c] += word_dot<VEC>(d, &wreg[q * VEC]);
                            }
                    };
                    if (nch >= T::CPS) chunks(std::integral_constant<int, T::CPS>{});
                    else if (nch == 1) chunks(std::integral_constant<int, 1>{});
                    else if constexpr (T::CPS == 4) {
                        if (nch == 2) chunks(std::integral_constant<int, 2>{});
                        else chunks(std::integral_constant<int, 3>{});
                    }
                    unsigned dep = 0; // the sums have consumed every word loaded from the stage
#pragma unroll
                    for (int c = 0; c < T::CPS; ++c) dep ^= dep_bits(acc[st * T::CPS + c]);
                    mbar_arrive_after_use(&empty[r2.s], lane, dep);
                    r2.advance(ns);
                }
            }
            };
            if (rows_left < R) tile(std::true_type{});
            else tile(std::false_type{});
        }
    }
    // ---- CTA partials: the four lanes of a group, then the sixteen warps in a fixed order ----------------------
    __syncthreads(); // every stage has been consumed: the stage memory is free for the partials
    double *hpart = reinterpret_cast<double *>(stages);                       // [16 warps][128 columns]
    double *npart_s = hpart + kConsumerWarps * kMaxRangeCols;                 // [2][16 warps]
    if (warp < kConsumerWarps) {
#pragma unroll
        for (int ch = 0; ch < kMaxChunks; ++ch) {
            double v = acc[ch];
            v += shfl_xor_f64(v, 1);
            v += shfl_xor_f64(v, 2);
            if ((lane & 3) == 0) hpart[warp * kMaxRangeCols + ch * kFGroups + (lane >> 2)] = v * PRE; // acc holds sums / PRE
        }
        ss = warp_sum(ss);
        am = warp_max(am);
        if (lane == 0) {
            npart_s[warp] = ss;
            npart_s[kConsumerWarps + warp] = am;
        }
    }
    __syncthreads();
    for (int col = tid; col < k; col += kOrthThreads) {
        double tsum = 0.0;
#pragma unroll
        for (int w = 0; w < kConsumerWarps; ++w) tsum += hpart[w * kMaxRangeCols + col];
        a.partials[(size_t)blockIdx.x * kLdp + col] = tsum;
    }
    if (tid == 0) {
        double tsum = 0.0, m = 0.0;
        for (int w = 0; w < kConsumerWarps; ++w) {
            tsum += npart_s[w];
            m = fmax(m, npart_s[kConsumerWarps + w]);
        }
        a.npart[blockIdx.x] = tsum;
        a.npart[kMaxGrid + blockIdx.x] = m;
    }
    if (!last_block_done(&ctl->tickets[0])) return;
    orth_finalize<PASS_UPD_DOT, Fm::SCALED>(a, k, reinterpret_cast<double *>(stages) + 4096); // scratch after the partials (32 KB in)
}

// ---- few vectors (k <= 8): no staging --------------------------------------------------------------------
// With at most eight basis vectors a row tile is a few KB and the staged kernel is bound by its
// per-tile round trips (multi-dot, n = 4.2e6: 50 us for k = 1..4, whatever the format).  Here a thread
// takes one 16-byte payload word of every vector plus the matching rows of w straight from global
// memory -- all loads of an iteration in flight together -- keeps the k words in registers for
// both sweeps of the fused kind, and the CTA reduces its partial sums through shuffles; the
// last-block-done final stage is the same as in orth_kernel.
constexpr int kSmallK = 8;

template <int FMT> __device__ __forceinline__ void decode_true(const uint4 &r, double (&d)[Fmt<FMT>::VEC])
{
    if constexpr (FMT == CBGMRES_FP64) {
        d[0] = __hiloint2double((int)r.y, (int)r.x);
        d[1] = __hiloint2double((int)r.w, (int)r.z);
    } else if constexpr (FMT == CBGMRES_FP32) {
        d[0] = (double)__uint_as_float(r.x);
        d[1] = (double)__uint_as_float(r.y);
        d[2] = (double)__uint_as_float(r.z);
        d[3] = (double)__uint_as_float(r.w);
    } else if constexpr (FMT == CBGMRES_INT32) {
        d[0] = (double)(int)r.x;
        d[1] = (double)(int)r.y;
        d[2] = (double)(int)r.z;
        d[3] = (double)(int)r.w;
    } else if constexpr (FMT == CBGMRES_FP16) {
        half2_cvt(r.x, d[0], d[1]);
        half2_cvt(r.y, d[2], d[3]);
        half2_cvt(r.z, d[4], d[5]);
        half2_cvt(r.w, d[6], d[7]);
    } else {
        i16x2_cvt(r.x, d[0], d[1]);
        i16x2_cvt(r.y, d[2], d[3]);
        i16x2_cvt(r.z, d[4], d[5]);
        i16x2_cvt(r.w, d[6], d[7]);
    }
}

template <int FMT, int KIND> __global__ void __launch_bounds__(kOrthThreads, 1) orth_small_kernel(const OrthArgs a)
{
    using Fm = Fmt<FMT>;
    constexpr int VEC = Fm::VEC, B = Fm::BYTES, NW = kOrthThreads / 32;
    constexpr bool HAS_UPD = KIND != PASS_DOT, HAS_DOT = KIND != PASS_UPD;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ double s_part[NW][kSmallK], s_nrm[2 * NW];
    Ctl *ctl = a.ctl;
    pdl_wait();
    pdl_launch_dependents();
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, k = a.k;
    const int stop_after = __ldcg(&ctl->stop_after), reorth_flag = __ldcg(&ctl->reorth_flag);
    double coef[kSmallK];
#pragma unroll
    for (int c = 0; c < kSmallK; ++c) coef[c] = (HAS_UPD && c < k) ? __ldcg(&a.hs[c]) : 0.0;
    if (a.mode == MODE_ORTH1 || a.mode == MODE_ORTH2) {
        if (a.step > stop_after) return;
        if (a.mode == MODE_ORTH2 && !reorth_flag) return;
    }
    double acc[kSmallK];
#pragma unroll
    for (int c = 0; c < kSmallK; ++c) acc[c] = 0.0;
    double ss = 0.0, am = 0.0;
    const unsigned char *V = static_cast<const unsigned char *>(a.V);
    const int64_t colb = a.ld * B, ngroups = a.n / VEC;
    for (int64_t g = (int64_t)blockIdx.x * kOrthThreads + tid; g < ngroups; g += (int64_t)gridDim.x * kOrthThreads) {
        uint4 raw[kSmallK];
#pragma unroll
        for (int c = 0; c < kSmallK; ++c)
            if (c < k) raw[c] = __ldg(reinterpret_cast<const uint4 *>(V + c * colb + g * 16));
        double wv[VEC];
#pragma unroll
        for (int v = 0; v < VEC; v += 2) {
            const double2 t = *reinterpret_cast<const double2 *>(a.w + g * VEC + v);
            wv[v] = t.x;
            wv[v + 1] = t.y;
        }
        if (HAS_UPD) {
            double p[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) p[v] = 0.0;
#pragma unroll
            for (int c = 0; c < kSmallK; ++c)
                if (c < k) {
                    double d[VEC];
                    decode_true<FMT>(raw[c], d);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) p[v] = fma(d[v], coef[c], p[v]);
                }
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                wv[v] -= p[v];
                ss = fma(wv[v], wv[v], ss);
                am = fmax(am, fabs(wv[v]));
            }
#pragma unroll
            for (int v = 0; v < VEC; v += 2) *reinterpret_cast<double2 *>(a.w + g * VEC + v) = make_double2(wv[v], wv[v + 1]);
        }
        if (HAS_DOT) {
#pragma unroll
            for (int c = 0; c < kSmallK; ++c)
                if (c < k) {
                    double d[VEC];
                    decode_true<FMT>(raw[c], d);
                    acc[c] += word_dot<VEC>(d, wv);
                }
        }
    }
    if (blockIdx.x == 0 && tid == 0) { // the last n mod VEC rows, one by one
        for (int64_t r = ngroups * VEC; r < a.n; ++r) {
            double wr = a.w[r];
            if (HAS_UPD) {
                double p = 0.0;
                for (int c = 0; c < k; ++c) p = fma(Fm::decode_one(V + c * colb, r), coef[c], p);
                wr -= p;
                a.w[r] = wr;
                ss = fma(wr, wr, ss);
                am = fmax(am, fabs(wr));
            }
            if (HAS_DOT)
                for (int c = 0; c < k; ++c) acc[c] = fma(Fm::decode_one(V + c * colb, r), wr, acc[c]);
        }
    }
    // ---- CTA partials: shuffles inside the warps, then the warps in a fixed order --------------------------
    if (HAS_DOT) {
#pragma unroll
        for (int c = 0; c < kSmallK; ++c) {
            const double t = warp_sum(acc[c]);
            if (lane == 0) s_part[warp][c] = t;
        }
    }
    if (HAS_UPD) {
        ss = warp_sum(ss);
        am = warp_max(am);
        if (lane == 0) {
            s_nrm[warp] = ss;
            s_nrm[NW + warp] = am;
        }
    }
    __syncthreads();
    if (HAS_DOT && tid < k) {
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < NW; ++q) t += s_part[q][tid];
        a.partials[(size_t)blockIdx.x * kLdp + tid] = t;
    }
    if (HAS_UPD && tid == 0) {
        double t = 0.0, m = 0.0;
#pragma unroll
        for (int q = 0; q < NW; ++q) {
            t += s_nrm[q];
            m = fmax(m, s_nrm[NW + q]);
        }
        a.npart[blockIdx.x] = t;
        a.npart[kMaxGrid + blockIdx.x] = m;
    }
    if (!last_block_done(&ctl->tickets[0])) return;
    orth_finalize<KIND, Fm::SCALED>(a, k, reinterpret_cast<double *>(smem));
}

// ---- launchers ---------------------------------------------------------------------------------------
namespace {

inline int fmt_bytes(int format) { return format == CBGMRES_FP64 ? 8 : (format == CBGMRES_FP32 || format == CBGMRES_INT32) ? 4 : 2; }
inline int fmt_max_seg_kb(int format) { return fmt_bytes(format) == 2 ? 2 : 4; } // F * VEC <= 16 rows per lane

inline int stages_for(int format, int seg_kb, bool has_upd)
{
    const int R = seg_kb * 1024 / fmt_bytes(format);
    const int ns = (kOrthSmemBytes - orth_fixed_smem(R, has_upd)) / kStageBytes;
    return ns > kMaxStages ? kMaxStages : ns;
}

// Column-segment size (KB) for a pass over k <= 128 columns; 0 = does not fit (fused kind only).
// forced != 0 pins the size (clamped to what the format allows) when that is feasible.
int choose_seg_kb(int format, int kind, int k, int64_t n, int forced)
{
    const int B = fmt_bytes(format);
    const int fmax = fmt_max_seg_kb(format);
    const int64_t per = ((n + kNumSMs - 1) / kNumSMs + 63) / 64 * 64; // rows per CTA on a full grid
    auto tile_stages = [&](int f) { return (k * f + 31) / 32; };      // a stage holds 32 / f columns
    auto feasible = [&](int f) {
        const int ns = stages_for(format, f, kind != PASS_DOT);
        return kind == PASS_UPD_DOT ? ns >= tile_stages(f) + 1 : ns >= 3;
    };
    if (forced) {
        const int f = forced > fmax ? fmax : forced;
        if (feasible(f)) return f;
    }
    for (int f = fmax; f >= 1; f >>= 1) {
        if (!feasible(f)) continue;
        // at least twelve row tiles per CTA: with fewer, pipeline ramp, tail and the one-tile imbalance of the
        // round-robin deal show (C2, n = 1e6, us per Arnoldi step at 6.6 / 13 / 26 tiles per CTA: fp32 182 / 169 / 172,
        // fp16 150 / 141 / -)
        if (f == 1 || (int64_t)f * 1024 / B * 12 <= per) return f;
    }
    return 0;
}

// ---- tensor maps: the basis as a 2D array [k columns][ceil(n*B/8) 8-byte words], box = 8 columns x
// (1 or 2 KB).  Rows beyond n*B bytes and columns beyond k are out of range: not fetched, read as zero.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

struct MapKey {
    const void *V = nullptr;
    int64_t ld = 0, n = 0;
    int bytes = 0, k = 0, inner = 0;
    bool operator==(const MapKey &o) const
    {
        return V == o.V && ld == o.ld && n == o.n && bytes == o.bytes && k == o.k && inner == o.inner;
    }
};

// One cached map per column count: inside a solve the same (V, k) comes back every restart cycle.
const CUtensorMap *basis_map(LaunchCtx *lc, const void *V, int64_t ld, int64_t n, int bytes, int k, int inner)
{
    struct Entry {
        MapKey key;
        CUtensorMap map;
    };
    static thread_local Entry cache[2][kMaxRangeCols + 1];
    Entry &e = cache[inner == 1024 ? 0 : 1][k];
    const MapKey key{V, ld, n, bytes, k, inner};
    if (e.key == key) return &e.map;
    EncodeTiledFn fn = encode_fn();
    if (!fn) {
        lc->orth_error = 999; // CUDA_ERROR_UNKNOWN: the driver has no cuTensorMapEncodeTiled
        return nullptr;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)((n * bytes + 7) / 8), (cuuint64_t)k};
    const cuuint64_t strides[1] = {(cuuint64_t)(ld * bytes)};
    const cuuint32_t box[2] = {(cuuint32_t)(inner / 8), (cuuint32_t)kChunkCols};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult rc = fn(&e.map, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, const_cast<void *>(V), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (rc != CUDA_SUCCESS) {
        lc->orth_error = (int)rc;
        e.key = MapKey{};
        return nullptr;
    }
    e.key = key;
    return &e.map;
}

// w as a 2D array [n / VEC groups][VEC doubles] with box [VEC x R / VEC] and the 32/64-byte swizzle
// (see wswz).  Only complete groups are in range; rows beyond them read as zero.
const CUtensorMap *w_map(LaunchCtx *lc, const double *w, int64_t n, int vec, int R)
{
    struct Entry {
        const double *w = nullptr;
        int64_t n = 0;
        int vec = 0, R = 0;
        CUtensorMap map;
    };
    static thread_local Entry cache[16];
    static thread_local int next = 0;
    for (Entry &e : cache)
        if (e.w == w && e.n == n && e.vec == vec && e.R == R) return &e.map;
    EncodeTiledFn fn = encode_fn();
    if (!fn) {
        lc->orth_error = 999;
        return nullptr;
    }
    Entry &e = cache[next];
    next = (next + 1) % 16;
    e.w = nullptr;
    const cuuint64_t groups = (cuuint64_t)(n / vec);
    const cuuint64_t dims[2] = {(cuuint64_t)vec, groups ? groups : 1};
    const cuuint64_t strides[1] = {(cuuint64_t)vec * 8};
    const cuuint32_t box[2] = {(cuuint32_t)vec, (cuuint32_t)(R / vec)};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult rc = fn(&e.map, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, const_cast<double *>(w), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, vec == 8 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_32B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (rc != CUDA_SUCCESS) {
        lc->orth_error = (int)rc;
        return nullptr;
    }
    e.w = w;
    e.n = n;
    e.vec = vec;
    e.R = R;
    return &e.map;
}

// The basis as the 3D array [ceil(n*B/128) segments of 128 bytes][k columns][16 words of 8 bytes] for
// orth_fused_kernel: box [16 x 8 columns x segs segments] with the 128-byte swizzle.  Needs ld*B % 128 == 0: the
// last, partial segment of a column then reads that column's own padding (masked by the kernel).
const CUtensorMap *basis_map3(LaunchCtx *lc, const void *V, int64_t ld, int64_t n, int bytes, int k, int segs)
{
    struct Entry {
        MapKey key;
        CUtensorMap map;
    };
    static thread_local Entry cache[2][kMaxRangeCols + 1];
    Entry &e = cache[segs == 8 ? 0 : 1][k];
    const MapKey key{V, ld, n, bytes, k, segs};
    if (e.key == key) return &e.map;
    EncodeTiledFn fn = encode_fn();
    if (!fn) {
        lc->orth_error = 999;
        return nullptr;
    }
    const cuuint64_t dims[3] = {16, (cuuint64_t)k, (cuuint64_t)((n * bytes + 127) / 128)};
    const cuuint64_t strides[2] = {(cuuint64_t)(ld * bytes), 128};
    const cuuint32_t box[3] = {16, (cuuint32_t)kFGroups, (cuuint32_t)segs};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult rc = fn(&e.map, CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, const_cast<void *>(V), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (rc != CUDA_SUCCESS) {
        lc->orth_error = (int)rc;
        e.key = MapKey{};
        return nullptr;
    }
    e.key = key;
    return &e.map;
}

inline int fused_stages(int format, int wpl)
{
    const int R = wpl * 1024 / fmt_bytes(format);
    const int ns = (kOrthSmemBytes - 1024 - ((ffixed_smem(R) + 1023) & ~1023)) / kStageBytes;
    return ns > kMaxStages ? kMaxStages : ns;
}
// words per lane and column (1 or 2, i.e. 1 or 2 KB column segments) for the row-mapped fused pass; 0 = not usable
int choose_fused_wpl(int format, int k, int64_t n, int64_t ld, int forced_seg_kb)
{
    const int B = fmt_bytes(format);
    if (B == 8 || k < 1 || k > kMaxRangeCols || (ld * B) % 128 != 0 || forced_seg_kb > 2) return 0;
    const int64_t per = ((n + kNumSMs - 1) / kNumSMs + 63) / 64 * 64;
    for (int wpl = 2; wpl >= 1; --wpl) {
        if (forced_seg_kb && wpl != forced_seg_kb) continue;
        if (wpl == 2 && B == 2 && !forced_seg_kb) continue; // 16 rows per lane: 96 registers do not hold them (spills)
        const int nst = (k * wpl + 31) / 32; // a stage holds 32 / wpl columns
        if (fused_stages(format, wpl) < nst + 1) continue;
        if (wpl == 1 || forced_seg_kb || (int64_t)wpl * 1024 / B * 12 <= per) return wpl; // at least twelve row tiles per CTA
    }
    return 0;
}

template <int FMT, int WPL> int launch_fused_inst(cudaStream_t s, const Scratch &sc, OrthArgs &a)
{
    using T = FTile<FMT, WPL>;
    static unsigned long long attr_set = 0;
    if (first_use_on_device(attr_set, sc.lc->device))
        cudaFuncSetAttribute(orth_fused_kernel<FMT, WPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, kOrthSmemBytes);
    const CUtensorMap *map = basis_map3(sc.lc, a.V, a.ld, a.n, T::B, a.k, T::SEGS);
    if (!map) return 0;
    a.nstages = fused_stages(FMT, WPL);
    a.interleave = 1;
    int64_t grid = (a.n + T::R - 1) / T::R;
    if (grid > kNumSMs) grid = kNumSMs;
    const size_t smem = 1024 + (size_t)((ffixed_smem(T::R) + 1023) & ~1023) + (size_t)a.nstages * kStageBytes;
    launch_chain(sc, "orth_fused_kernel", orth_fused_kernel<FMT, WPL>, dim3((unsigned)grid), dim3(kOrthThreads), smem, s, a, *map);
    return 1;
}

template <int FMT> int launch_fused_f(cudaStream_t s, const Scratch &sc, OrthArgs &a, int wpl)
{
    return wpl == 2 ? launch_fused_inst<FMT, 2>(s, sc, a) : launch_fused_inst<FMT, 1>(s, sc, a);
}

int launch_fused(cudaStream_t s, const Scratch &sc, int format, OrthArgs &a, int wpl)
{
    switch (format) {
    case CBGMRES_FP32: return launch_fused_f<CBGMRES_FP32>(s, sc, a, wpl);
    case CBGMRES_FP16: return launch_fused_f<CBGMRES_FP16>(s, sc, a, wpl);
    case CBGMRES_INT32: return launch_fused_f<CBGMRES_INT32>(s, sc, a, wpl);
    case CBGMRES_INT16: return launch_fused_f<CBGMRES_INT16>(s, sc, a, wpl);
    default: return 0;
    }
}

template <int FMT, int F, int KIND> int launch_inst(cudaStream_t s, const Scratch &sc, OrthArgs &a)
{
    using T = Tile<FMT, F>;
    a.interleave = sc.lc->interleave != 1; // measured: the shared sliding window wins for every segment size (fp64 k = 100: 6.46 -> 6.75 TB/s)
    static unsigned long long attr_set = 0; // the opt-in to 225 KB of dynamic shared memory is per device
    if (first_use_on_device(attr_set, sc.lc->device))
        cudaFuncSetAttribute(orth_kernel<FMT, F, KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, kOrthSmemBytes);
    const CUtensorMap *map = basis_map(sc.lc, a.V, a.ld, a.n, T::B, a.k, T::BOX_INNER);
    if (!map) return 0;
    const CUtensorMap *wm = (T::VEC == 2) ? map : w_map(sc.lc, a.w, a.n, T::VEC, T::R); // fp64: linear w tiles, map unused
    if (!wm) return 0;
    a.nstages = stages_for(FMT, F, KIND != PASS_DOT);
    int64_t grid = (a.n + 63) / 64;
    if (grid > kNumSMs) grid = kNumSMs;
    const size_t smem = (size_t)orth_fixed_smem(T::R, KIND != PASS_DOT) + (size_t)a.nstages * T::STAGE;
    launch_chain(sc, "orth_kernel", orth_kernel<FMT, F, KIND>, dim3((unsigned)grid), dim3(kOrthThreads), smem, s, a, *map, *wm);
    return 1;
}

constexpr int kSmallSmemBytes = 17 * 1024; // the final stage's scratch ([16][128] doubles)

template <int KIND> int launch_small(cudaStream_t s, const Scratch &sc, int format, OrthArgs &a)
{
    const int64_t groups = a.n / (16 / fmt_bytes(format));
    int64_t grid = (groups + kOrthThreads - 1) / kOrthThreads;
    if (grid > kNumSMs) grid = kNumSMs;
    if (grid < 1) grid = 1;
    const dim3 g((unsigned)grid), b(kOrthThreads);
    switch (format) {
    case CBGMRES_FP64: launch_chain(sc, "orth_small_kernel", orth_small_kernel<CBGMRES_FP64, KIND>, g, b, kSmallSmemBytes, s, a); break;
    case CBGMRES_FP32: launch_chain(sc, "orth_small_kernel", orth_small_kernel<CBGMRES_FP32, KIND>, g, b, kSmallSmemBytes, s, a); break;
    case CBGMRES_FP16: launch_chain(sc, "orth_small_kernel", orth_small_kernel<CBGMRES_FP16, KIND>, g, b, kSmallSmemBytes, s, a); break;
    case CBGMRES_INT32: launch_chain(sc, "orth_small_kernel", orth_small_kernel<CBGMRES_INT32, KIND>, g, b, kSmallSmemBytes, s, a); break;
    case CBGMRES_INT16: launch_chain(sc, "orth_small_kernel", orth_small_kernel<CBGMRES_INT16, KIND>, g, b, kSmallSmemBytes, s, a); break;
    default: return 0;
    }
    return 1;
}
// k <= 8, column count known on the host, segment size not pinned by the caller, 16-byte aligned columns
inline bool use_small(const OrthArgs &a, int format, int forced_seg_kb)
{
    return a.k <= kSmallK && !a.d_k && forced_seg_kb == 0 && (a.ld * fmt_bytes(format)) % 16 == 0 &&
           reinterpret_cast<uintptr_t>(a.V) % 16 == 0 && reinterpret_cast<uintptr_t>(a.w) % 16 == 0;
}

template <int FMT, int KIND> int launch_f(cudaStream_t s, const Scratch &sc, OrthArgs &a, int seg_kb)
{
    constexpr int VEC = Fmt<FMT>::VEC;
    switch (seg_kb) {
    case 1: return launch_inst<FMT, 1, KIND>(s, sc, a);
    case 2: return launch_inst<FMT, 2, KIND>(s, sc, a);
    case 4:
        if constexpr (VEC <= 4) return launch_inst<FMT, 4, KIND>(s, sc, a);
        return 0;
    default: return 0;
    }
}

template <int KIND> int launch_fmt(cudaStream_t s, const Scratch &sc, int format, OrthArgs &a, int seg_kb)
{
    switch (format) {
    case CBGMRES_FP64: return launch_f<CBGMRES_FP64, KIND>(s, sc, a, seg_kb);
    case CBGMRES_FP32: return launch_f<CBGMRES_FP32, KIND>(s, sc, a, seg_kb);
    case CBGMRES_FP16: return launch_f<CBGMRES_FP16, KIND>(s, sc, a, seg_kb);
    case CBGMRES_INT32: return launch_f<CBGMRES_INT32, KIND>(s, sc, a, seg_kb);
    case CBGMRES_INT16: return launch_f<CBGMRES_INT16, KIND>(s, sc, a, seg_kb);
    default: return 0;
    }
}

OrthArgs base_args(const Scratch &sc, const BasisView &b, int64_t n, int mode, int step)
{
    OrthArgs a{};
    a.V = b.V;
    a.ld = b.ld;
    a.scales = b.scales;
    a.n = n;
    a.ctl = sc.ctl;
    a.partials = sc.partials;
    a.npart = sc.npart;
    a.mode = mode;
    a.step = step;
    a.last_range = 1;
    return a;
}

} // namespace


// S2 (and S2' when the fused pass does not fit): ranges of at most 128 columns per launch.
int launch_multidot(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const double *w,
                    double *h_out, double *hs_out, int mode, int step, int seg_kb)
{
    int launches = 0;
    const int64_t col_bytes = b.ld * fmt_bytes(b.format);
    for (int c0 = 0; c0 < k; c0 += kMaxRangeCols) {
        const int kk = (k - c0 < kMaxRangeCols) ? k - c0 : kMaxRangeCols;
        OrthArgs a = base_args(sc, b, n, mode, step);
        a.dir = 0; // dot forwards, first update backwards, second update forwards: each pass starts where the previous one ended
        a.V = static_cast<const char *>(b.V) + (int64_t)c0 * col_bytes;
        a.scales = b.scales ? b.scales + c0 : nullptr;
        a.w = const_cast<double *>(w);
        a.k = kk;
        a.h_out = h_out + c0;
        a.hs_out = hs_out ? hs_out + c0 : nullptr;
        a.last_range = (c0 + kMaxRangeCols >= k);
        if (use_small(a, b.format, seg_kb)) launches += launch_small<PASS_DOT>(s, sc, b.format, a);
        else launches += launch_fmt<PASS_DOT>(s, sc, b.format, a, choose_seg_kb(b.format, PASS_DOT, kk, n, seg_kb));
    }
    return launches;
}

// S3 / S3' / the x update of l.17 (d_k != null: the column count lives on the device, k is its bound).
int launch_update(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const int *d_k,
                  const double *hs, double *w, int mode, int step, int seg_kb)
{
    int launches = 0;
    const int64_t col_bytes = b.ld * fmt_bytes(b.format);
    for (int c0 = 0; c0 < k; c0 += kMaxRangeCols) {
        const int kk = (k - c0 < kMaxRangeCols) ? k - c0 : kMaxRangeCols;
        OrthArgs a = base_args(sc, b, n, mode, step);
        a.dir = (mode == MODE_ORTH1) ? 1 : 0; // dot forwards, first update backwards, second update forwards: each pass starts where the previous one ended
        a.V = static_cast<const char *>(b.V) + (int64_t)c0 * col_bytes;
        a.hs = hs + c0;
        a.d_k = d_k;
        a.c0 = c0;
        a.w = w;
        a.k = kk;
        a.last_range = (c0 + kMaxRangeCols >= k);
        if (use_small(a, b.format, seg_kb)) launches += launch_small<PASS_UPD>(s, sc, b.format, a);
        else launches += launch_fmt<PASS_UPD>(s, sc, b.format, a, choose_seg_kb(b.format, PASS_UPD, kk, n, seg_kb));
    }
    return launches;
}

bool update_multidot_fits(int format, int k, int seg_kb)
{
    return k >= 1 && k <= kMaxRangeCols && choose_seg_kb(format, PASS_UPD_DOT, k, 1 << 30, seg_kb) != 0;
}

int launch_update_multidot(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const double *hs,
                           double *w, double *h_out, double *hs_out, int mode, int step, int seg_kb)
{
    if (!update_multidot_fits(b.format, k, seg_kb)) return 0;
    OrthArgs a = base_args(sc, b, n, mode, step);
        a.dir = (mode == MODE_HOOK) ? 0 : 1; // dot forwards, first update backwards, second update forwards: each pass starts where the previous one ended
    a.hs = hs;
    a.w = w;
    a.k = k;
    a.h_out = h_out;
    a.hs_out = hs_out;
    if (use_small(a, b.format, seg_kb)) return launch_small<PASS_UPD_DOT>(s, sc, b.format, a);
    // warps own rows, shuffle reduction (orth_fused_kernel): measured equal to the column-mapped kind within 1-3 % at every
    // k (n = 4.2e6: fp16 k = 32 / 64 / 128: 124 / 192 / 290 us against 130 / 177 / 294; fp32 136 / 222 / 396 against 145 / 224 / 380),
    // a little ahead for the 16-bit formats inside the solves (C2 int16 53 against 57 us), a little behind for the 32-bit ones
    if (sc.lc->fused_rows == 1 || (sc.lc->fused_rows == 2 && fmt_bytes(b.format) == 2)) {
        const int wpl = choose_fused_wpl(b.format, k, n, b.ld, seg_kb);
        if (wpl) return launch_fused(s, sc, b.format, a, wpl);
    }
    return launch_fmt<PASS_UPD_DOT>(s, sc, b.format, a, choose_seg_kb(b.format, PASS_UPD_DOT, k, n, seg_kb));
}

} // namespace cbg
