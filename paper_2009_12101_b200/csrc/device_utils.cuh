// device_utils.cuh -- storage-format traits (decode in registers), encoders, warp/block
// reductions and the last-block-done ticket used by every reduction kernel.
#pragma once
#include "internal.cuh"

namespace cbg {

// ---- 128-bit streaming loads -------------------------------------------------------------------
// Basis payloads are read once per kernel: bypass L1 allocation, keep the default L2 policy so
// that the update pass can still find the multi-dot pass's lines in the 126 MB L2.
__device__ __forceinline__ uint4 ldg_stream128(const void *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

// ---- widening to binary64 without the conversion pipe ---------------------------------------------
// cvt.f64.f32 / cvt.f64.s32 issue at a quarter of the fp64 FMA rate; at 2 bytes per entry the basis
// delivers ~11 entries per clock and SM, which that pipe cannot convert.  These build a binary64 bit
// pattern with integer ops.  For the floating-point formats the pattern is the value times the bias
// difference 2^-S (S = 896 for binary32, 1008 for binary16; a subnormal input becomes a binary64
// subnormal, which the fp64 pipe takes at full speed); the passes multiply the OTHER operand of
// every product (the tile of w, the coefficients h_c) by 2^(S/2) once and the result by 2^(S/2)
// once, so no per-entry multiply is left.  Scaling by a power of two commutes with rounding (no
// intermediate leaves the normal range: that would need abs(value) < 2^-518 or >= 2^520), so the
// results are bit-identical to widening first.  Fixed point: 2^52 + offset + q is exact in the
// binade of 2^52; one fp64 subtraction removes the offset.
// (Define CBG_DECODE_CVT to get the plain conversions back.)
#ifdef CBG_DECODE_CVT
constexpr double kPreF32 = 1.0, kPreF16 = 1.0, kPreF16Even = 1.0;
__device__ __forceinline__ double f32_bits_to_raw(unsigned f) { return (double)__uint_as_float(f); }
__device__ __forceinline__ double i32_to_double(int q) { return (double)q; }
// F2F.F64.F16 / I2F.F64.S16 take either half of a 32-bit register: one instruction per entry
__device__ __forceinline__ void half2_to_raw(unsigned w, double &lo, double &hi)
{
    asm("{.reg .b16 l, h; mov.b32 {l, h}, %2; cvt.f64.f16 %0, l; cvt.f64.f16 %1, h;}" : "=d"(lo), "=d"(hi) : "r"(w));
}
__device__ __forceinline__ void i16x2_to_doubles(unsigned w, double &lo, double &hi)
{
    asm("{.reg .b16 l, h; mov.b32 {l, h}, %2; cvt.rn.f64.s16 %0, l; cvt.rn.f64.s16 %1, h;}" : "=d"(lo), "=d"(hi) : "r"(w));
}
#else
constexpr double kPreF32 = 0x1p448, kPreF16 = 0x1p504;
// binary32 -> value * 2^-896: sign | exponent field | 23 fraction bits at the top of the binary64 fraction.
__device__ __forceinline__ double f32_bits_to_raw(unsigned f)
{
    const unsigned hi = (unsigned)((int)f >> 3) & 0x8FFFFFFFu;
    return __hiloint2double((int)hi, (int)(f << 29));
}
// int32 -> binary64: 2^52 + 2^31 + q, minus the offset.
__device__ __forceinline__ double i32_to_double(int q)
{
    return __hiloint2double(0x43300000, q ^ (int)0x80000000) - 4503601774854144.0;
}
// Two 16-bit entries per 32-bit payload word, MIXED widening (CBG_DECODE_MIXED, default): the LOW half goes
// through the conversion pipe (F2F.F64.F16 / I2F.F64.S16 read either half of a register: one instruction,
// 16 per clock and SM), the HIGH half through the integer pipes (arithmetic shift + mask in place, no
// left shift needed).  A 16-bit pass at the HBM rate delivers 11.2 entries per clock and SM: all of them
// through the conversion pipe would saturate it, all of them through the integer pipes cost 3.8 issue
// slots per entry (measured from ncu's instruction counts); half and half is 2.75.  For binary16 the two
// halves then carry different powers of two -- the low half is the true value, the high half value * 2^-1008
// -- so the OTHER operand of every product carries 2^-504 on even rows and 2^+504 on odd rows
// (Fmt::PRE_EVEN / Fmt::PRE): every product is value * operand * 2^-504 exactly as before, bit for bit.
#ifndef CBG_DECODE_MIXED
#define CBG_DECODE_MIXED 1
#endif
#if CBG_DECODE_MIXED
constexpr double kPreF16Even = 0x1p-504;
__device__ __forceinline__ void half2_to_raw(unsigned w, double &lo, double &hi)
{
    asm("{.reg .b16 l, h; mov.b32 {l, h}, %1; cvt.f64.f16 %0, l;}" : "=d"(lo) : "r"(w));
    const unsigned h1 = (unsigned)((int)w >> 6) & 0x81FFFC00u;
    hi = __hiloint2double((int)h1, 0);
}
__device__ __forceinline__ void i16x2_to_doubles(unsigned w, double &lo, double &hi)
{
    asm("{.reg .b16 l, h; mov.b32 {l, h}, %1; cvt.rn.f64.s16 %0, l;}" : "=d"(lo) : "r"(w));
    hi = __hiloint2double(0x43300000, (int)((w >> 16) ^ 0x8000u)) - 4503599627403264.0; // 2^52 + 32768 + q, minus the offset
}
#else
constexpr double kPreF16Even = kPreF16;
// two binary16 -> values * 2^-1008.
__device__ __forceinline__ void half2_to_raw(unsigned w, double &lo, double &hi)
{
    const unsigned h1 = (unsigned)((int)w >> 6) & 0x81FFFC00u;
    const unsigned h0 = (unsigned)((int)(w << 16) >> 6) & 0x81FFFC00u;
    lo = __hiloint2double((int)h0, 0);
    hi = __hiloint2double((int)h1, 0);
}
// two int16 -> binary64: flip both sign bits at once (q + 32768 as an unsigned 16-bit field), then
// 2^52 + 32768 + q minus the offset.
__device__ __forceinline__ void i16x2_to_doubles(unsigned w, double &lo, double &hi)
{
    const unsigned u = w ^ 0x80008000u;
    lo = __hiloint2double(0x43300000, (int)(u & 0xFFFFu)) - 4503599627403264.0;
    hi = __hiloint2double(0x43300000, (int)(u >> 16)) - 4503599627403264.0;
}
#endif
#endif

// ---- storage formats ----------------------------------------------------------
// VEC = entries per 128-bit load.  decode() widens one 128-bit payload word to VEC fp64 values
// WITHOUT the per-vector scale: the fixed-point scale sigma_c is folded into the coefficient
// (h_c = sigma_c * sum q w ; w -= sum q (sigma_c h_c)), so the "one multiplication per element"
// of PAPER.md:181 disappears from the inner loops.
template <int FMT> struct Fmt;

template <> struct Fmt<CBGMRES_FP64> {
    static constexpr int VEC = 2, BYTES = 8;
    static constexpr bool SCALED = false;
    static constexpr double PRE = 1.0; // decode() yields value / PRE^2 (see "widening" above)
    static constexpr double PRE_EVEN = 1.0; // ... on even entries value / (PRE * PRE_EVEN) (mixed widening of binary16)
    __device__ static __forceinline__ void decode(const uint4 &r, double (&d)[VEC])
    {
        d[0] = __hiloint2double((int)r.y, (int)r.x);
        d[1] = __hiloint2double((int)r.w, (int)r.z);
    }
    __device__ static __forceinline__ double decode_one(const void *col, int64_t i) { return ((const double *)col)[i]; }
};

template <> struct Fmt<CBGMRES_FP32> {
    static constexpr int VEC = 4, BYTES = 4;
    static constexpr bool SCALED = false;
    static constexpr double PRE = kPreF32;
    static constexpr double PRE_EVEN = kPreF32; // (mixed widening measured no faster for the 32-bit formats: fp32 fused k = 100 384 against 333 us)
    __device__ static __forceinline__ void decode(const uint4 &r, double (&d)[VEC])
    {
        d[0] = f32_bits_to_raw(r.x);
        d[1] = f32_bits_to_raw(r.y);
        d[2] = f32_bits_to_raw(r.z);
        d[3] = f32_bits_to_raw(r.w);
    }
    __device__ static __forceinline__ double decode_one(const void *col, int64_t i)
    {
        return (double)((const float *)col)[i];
    }
};



template <> struct Fmt<CBGMRES_FP16> {
    static constexpr int VEC = 8, BYTES = 2;
    static constexpr bool SCALED = false;
    static constexpr double PRE = kPreF16;
    static constexpr double PRE_EVEN = kPreF16Even;
    __device__ static __forceinline__ void decode(const uint4 &r, double (&d)[VEC])
    {
        half2_to_raw(r.x, d[0], d[1]);
        half2_to_raw(r.y, d[2], d[3]);
        half2_to_raw(r.z, d[4], d[5]);
        half2_to_raw(r.w, d[6], d[7]);
    }
    __device__ static __forceinline__ double decode_one(const void *col, int64_t i)
    {
        return (double)__half2float(((const __half *)col)[i]);
    }
};

template <> struct Fmt<CBGMRES_INT32> {
    static constexpr int VEC = 4, BYTES = 4;
    static constexpr bool SCALED = true;
    static constexpr double PRE = 1.0;
    static constexpr double PRE_EVEN = 1.0;
    __device__ static __forceinline__ void decode(const uint4 &r, double (&d)[VEC])
    {
        d[0] = i32_to_double((int)r.x);
        d[1] = i32_to_double((int)r.y);
        d[2] = i32_to_double((int)r.z);
        d[3] = i32_to_double((int)r.w);
    }
    __device__ static __forceinline__ double decode_one(const void *col, int64_t i)
    {
        return (double)((const int32_t *)col)[i];
    }
};

template <> struct Fmt<CBGMRES_INT16> {
    static constexpr int VEC = 8, BYTES = 2;
    static constexpr bool SCALED = true;
    static constexpr double PRE = 1.0;
    static constexpr double PRE_EVEN = 1.0;
    __device__ static __forceinline__ void decode(const uint4 &r, double (&d)[VEC])
    {
        i16x2_to_doubles(r.x, d[0], d[1]);
        i16x2_to_doubles(r.y, d[2], d[3]);
        i16x2_to_doubles(r.z, d[4], d[5]);
        i16x2_to_doubles(r.w, d[6], d[7]);
    }
    __device__ static __forceinline__ double decode_one(const void *col, int64_t i)
    {
        return (double)((const int16_t *)col)[i];
    }
};

// ---- encoders (bit-exact functions of the fp64 input; readings Q6-Q8) ----------------
// s = max_int / a for the fixed-point formats (unused otherwise).
template <int FMT> __device__ __forceinline__ unsigned enc_bits(double v, double s);
template <> __device__ __forceinline__ unsigned enc_bits<CBGMRES_FP32>(double v, double)
{
    return __float_as_uint(__double2float_rn(v)); // cvt.rn.f32.f64, no .ftz: gradual underflow
}
template <> __device__ __forceinline__ unsigned enc_bits<CBGMRES_FP16>(double v, double)
{
    return (unsigned)__half_as_ushort(__double2half(v)); // cvt.rn.f16.f64: ONE rounding
}
template <> __device__ __forceinline__ unsigned enc_bits<CBGMRES_INT32>(double v, double s)
{
    int q = __double2int_rn(__dmul_rn(v, s)); // ties to even; saturates
    q = max(q, -2147483647);                  // symmetric clamp (reading Q6)
    return (unsigned)q;
}
template <> __device__ __forceinline__ unsigned enc_bits<CBGMRES_INT16>(double v, double s)
{
    int q = __double2int_rn(__dmul_rn(v, s));
    q = min(max(q, -32767), 32767);
    return (unsigned)q & 0xFFFFu;
}

template <int FMT> __device__ __forceinline__ double fmt_maxint()
{
    return FMT == CBGMRES_INT32 ? 2147483647.0 : 32767.0;
}

// ---- reductions ---------------------------------------------------------------------------------
__device__ __forceinline__ double shfl_xor_f64(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += shfl_xor_f64(v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, shfl_xor_f64(v, o));
    return v;
}

// Transposing butterfly: every lane holds N partial sums (one per column); afterwards lane L with
// (L % (32/N)) == 0 holds the warp total of column butterfly_col<N>(L).  N + log2(32/N) - 1
// shuffles instead of 5 N.  Summation order is fixed, so results are reproducible.
template <int N, int OFF> __device__ __forceinline__ double butterfly_rec(double (&a)[N], int lane)
{
    if constexpr (N == 1) {
        double v = a[0];
#pragma unroll
        for (int o = OFF; o > 0; o >>= 1) v += shfl_xor_f64(v, o);
        return v;
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
        return butterfly_rec<H, OFF / 2>(b, lane);
    }
}

// Column held by lane L after butterfly_rec<N,16>: the top log2(N) bits of L, MSB first.
template <int N> __device__ __forceinline__ int butterfly_col(int lane)
{
    int col = 0, off = 16;
#pragma unroll
    for (int h = N / 2; h >= 1; h >>= 1) {
        if (lane & off) col += h;
        off >>= 1;
    }
    return col;
}
template <int N> __device__ __forceinline__ bool butterfly_owner(int lane) { return (lane & (32 / N - 1)) == 0; }

// Last-block-done ticket: returns true in every thread of the CTA that arrives last.  Partials
// written before the call are visible to that CTA.  The counter is reset for the next launch.
__device__ __forceinline__ bool last_block_done(unsigned *ticket)
{
    __shared__ int s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last) *ticket = 0u;
    }
    __syncthreads();
    if (s_last) __threadfence();
    return s_last != 0;
}

// ---- mbarrier / bulk-copy primitives (PTX) --------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LAB_DONE;\n"
        "bra LAB_WAIT;\n"
        "LAB_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 1D bulk copy global -> shared (TMA engine), bytes a multiple of 16, both addresses 16-byte aligned.
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// The same with an L2 cache policy (createpolicy): the matrix stream of the SpMV is marked evict-first so
// that it does not push the basis and the vectors out of the 126 MB L2 between two Gram-Schmidt passes.
__device__ __forceinline__ void bulk_g2s_hint(void *dst_smem, const void *src, uint32_t bytes, uint64_t *bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
                 : "memory");
}

// ---- programmatic dependent launch ------------------------------------------------------------------
// The kernels of an Arnoldi step form a chain on one stream, each 10-100 us long.  Launched with
// the programmatic-stream-serialisation attribute, the next kernel's CTAs are scheduled while the
// tail of the previous one (its last-block-done final stage) is still running, and park in
// griddepcontrol.wait until that grid has completed and flushed; nothing produced by a predecessor
// is read before the wait.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Launch on stream s as a link of the step chain (programmatic stream serialisation unless the handle's
// "pdl" option is off).  A failed launch is recorded in the handle's LaunchCtx with the kernel's name
// (the first failure wins); the solver checks it after every enqueued step.
template <class... KArgs, class... Args>
inline cudaError_t launch_chain(const Scratch &sc, const char *name, void (*kernel)(KArgs...), dim3 grid, dim3 block,
                                size_t smem, cudaStream_t s, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = sc.lc->use_pdl ? 1 : 0;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
    if (e != cudaSuccess && sc.lc->launch_error == cudaSuccess) {
        sc.lc->launch_error = e;
        sc.lc->launch_kernel = name;
    }
    return e;
}

// Hand a shared-memory slot back to the producer (arrive on its "empty" mbarrier) -- but only once
// the values loaded from it have been USED by every lane: loads that have merely been issued can be
// overtaken by the producer's next TMA write into the slot (seen as wrong inner products; a
// CTA-scope MEMBAR.SC also closes the window but costs ~400 cycles per release).  `dep` must be
// computed from results that consumed every load from the slot; the warp vote needs it from all 32
// lanes and its result is an input of the arrive, so neither can be scheduled before the uses.
// Why this is sufficient (there is no racecheck on this pool, so the argument is written down):
//  (1) Hardware: an LDS whose result has been consumed by an arithmetic instruction has completed -- the
//      scoreboard releases the consumer only when the loaded value is in the register file -- so once `dep` exists,
//      no read of the slot by this lane is still in flight.
//  (2) Compiler: `dep` is data-dependent on every value loaded from the slot (the callers fold one accumulator per
//      128-bit load into it); the ballot's predicate depends on `dep`, the ballot needs all 32 lanes, and its result `b`
//      is an INPUT operand of the asm volatile arrive ("memory" clobber): the arrive cannot be hoisted above the
//      ballot, nor the ballot above the last use, in any lane.  (The comparison constant is a NaN pattern no
//      accumulator produces; the branch is never taken -- it only keeps the dependency alive.)
//  (3) Memory model: mbarrier.arrive has release semantics at CTA scope, the producer's try_wait acquires; the
//      producer's next cp.async.bulk into the slot is issued after that wait, so it is ordered after the reads of (1).
//      The reads are generic-proxy reads, the refill an async-proxy write: a write-after-read across the proxies needs
//      no proxy fence (only generic-proxy WRITES to the slot do, which is why the ragged w tile, patched by hand, issues
//      fence.proxy.async before its arrive).
// Regression tests: test_multidot_many_tiles_per_cta_repeats_bitwise, test_full_size_c2_solve_is_bitwise_repeatable.
__device__ __forceinline__ unsigned dep_bits(double x) { return (unsigned)__double2hiint(x); }
__device__ __forceinline__ void mbar_arrive_after_use(uint64_t *bar, int lane, unsigned dep)
{
    const unsigned b = __ballot_sync(0xffffffffu, dep != 0x7ff1a5a5u);
    if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0]; // after %1" ::"r"(smem_u32(bar)), "r"(b) : "memory");
}

// Position in a ring of shared-memory stages and the parity of its mbarriers.
struct Ring {
    int s = 0;
    uint32_t ph = 0;
    __device__ __forceinline__ void advance(int ns)
    {
        if (++s == ns) {
            s = 0;
            ph ^= 1u;
        }
    }
};

} // namespace cbg
