/*
 * zmc_device.cuh -- device code of the fused sampling kernel (sm_100a).
 *
 * Philox4x32-10 -> word -> point -> integrand -> FP64 sum, all in registers: no sample is ever
 * written to memory ("produce the random number at the time when using it").
 * One warp processes one work item = (cell, trial, sample chunk); a persistent grid pulls items
 * from a device counter whose bound was written by the previous level's control kernels, so the
 * host enqueues all levels up front.
 *
 * What bounds it: the 32x32->64-bit multiplies of Philox, IMAD.WIDE.U32, run
 * only on the FMA-heavy pipe (4 clocks per warp-instruction), and next to them nothing issues for
 * free. So the kernel is built to issue as few other instructions as possible: two samples per
 * packed FP32 instruction (FFMA2/FADD2/FMUL2), round keys in uniform registers when the launch has
 * one key (UKEY), 2 or 4 sample groups per loop trip, per-dimension choices in ZmcTune.
 *
 * This file is self-contained (no #include) because it is compiled twice: ahead of time by nvcc
 * for the built-in integrands (zmc_inst_*.cu) and at run time by NVRTC for user integrands and
 * for dimensions without a pre-compiled instance (zmc_lib.cu embeds this text).
 * It shares nothing with oracle/: the operation sequences below restate DESIGN.md R1-R8.
 *
 * Compile with --fmad=false: every fused multiply-add here is written explicitly.
 */
#ifndef ZMC_DEVICE_CUH
#define ZMC_DEVICE_CUH

typedef unsigned int zu32;
typedef unsigned long long zu64;
typedef int zi32;

#define ZMC_DEV_MAX_DIM 16
#define ZMC_HAS_TPI 1
#ifndef ZMC_BLOCK_THREADS
#define ZMC_BLOCK_THREADS 128
#endif

/* integrand ids / precision / math mode: values mirror include/zmc.h (checked by static_assert in zmc_lib.cu) */
#define ZMC_ID_CONST 0
#define ZMC_ID_LINEAR 1
#define ZMC_ID_SIN_SUM 2
#define ZMC_ID_EXP_QUAD 3
#define ZMC_ID_USER 100
#define ZMC_PREC_F64 0
#define ZMC_PREC_F32 1
#define ZMC_MODE_EXACT 0
#define ZMC_MODE_FAST 1

/* One per level (index 1..L) in device memory. Written by the previous level's control kernels
 * (level 1: by the init kernel); read by this level's kernels. */
struct ZmcLevelInfo {
    zu64 n_groups;      /* parents = sibling groups at this level */
    zu64 n_cells;       /* n_groups * k */
    zu64 n_items;       /* n_cells * (T / trials_per_item) * n_chunks work items */
    zu64 work_ctr;      /* the persistent grid's item counter */
    zu64 n_flagged;     /* cells with s > tau */
    zu64 n_refined;     /* flagged cells passed on (after budget and capacity) */
    zu32 n_chunks;      /* sample chunks per (cell, trial) unit */
    zu32 chunk_groups;  /* sample groups per chunk */
    zu32 trials_per_item; /* 1, or T on levels with many cells: one warp takes all trials of a cell, so that the item decoding
                             and the cell geometry are paid once per cell instead of once per trial (n_chunks == 1 then) */
    zu32 reserved;
    /* single-launch path only (zmc_tree.cuh): %globaltimer (ns) as block 0 passes the level's grid barriers -- level begun,
     * sampling done, statistics/thresholds done, control done: what zmc_stats reports as sample_ms / control_ms there */
    zu64 t_mark[4];
};

struct ZmcSampleArgs {
    const zu32* par_inst;    /* [G] instance of each parent */
    const zu64* par_plo;     /* [G] parent path, low 64 bits */
    const zu32* par_phi;     /* [G] parent path, bits 64..79 */
    const zu32* par_coord;   /* [d * par_stride + G] parent integer coordinates */
    zu64 par_stride;
    ZmcLevelInfo* info;      /* this level's */
    double* partial;         /* [item] FP64 partial sums, item = (cell*T + trial)*n_chunks + chunk */
    double* partial_q;       /* [item] FP64 partial sums of f^2 (SQ kernels only: R13) */
    const zu32* keys;        /* [instance][2] derived Philox keys (R3) */
    const double* params;    /* [instance][ppi] */
    const float* params_f32; /* the same rounded to FP32 (user integrands) */
    zi32 ppi;
    zu32 g, T, level;
    zu64 k;
    zu64 N;
    double lower[ZMC_DEV_MAX_DIM];
    double width[ZMC_DEV_MAX_DIM];   /* cell width at this level, (upper-lower)/g^level (R2) */
    zu32 ukey[2];                    /* UKEY kernels (n_instances == 1): the one derived key, read from the constant bank */
};

/* ------------------------------------------------------------------ R1: Philox4x32-10 */
/* Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11).
 * round: (hi0,lo0) = M0*c0 ; (hi1,lo1) = M1*c2 ; c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0) ; k += W.
 * Each round is 2 IMAD.WIDE.U32 + 2 LOP3 in SASS; the ten key values are loop-invariant. */
#define ZMC_PHILOX_M0 0xD2511F53u
#define ZMC_PHILOX_M1 0xCD9E8D57u
#define ZMC_PHILOX_W0 0x9E3779B9u
#define ZMC_PHILOX_W1 0xBB67AE85u

struct ZmcKeySchedule {
    zu32 k0[10], k1[10];
    __device__ __forceinline__ void init(zu32 key0, zu32 key1) {
#pragma unroll
        for (int r = 0; r < 10; ++r) { k0[r] = key0 + (zu32)r * ZMC_PHILOX_W0; k1[r] = key1 + (zu32)r * ZMC_PHILOX_W1; }
    }
};

__device__ __forceinline__ void zmc_philox(zu32 c0, zu32 c1, zu32 c2, zu32 c3, const ZmcKeySchedule& ks, zu32* out) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const zu64 p0 = (zu64)c0 * (zu64)ZMC_PHILOX_M0;
        const zu64 p1 = (zu64)c2 * (zu64)ZMC_PHILOX_M1;
        const zu32 n0 = (zu32)(p1 >> 32) ^ c1 ^ ks.k0[r];
        const zu32 n2 = (zu32)(p0 >> 32) ^ c3 ^ ks.k1[r];
        c1 = (zu32)p1;
        c3 = (zu32)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* The same with the first round's product M0*c0 supplied by the caller: consecutive call indices differ by 1,
 * so their products differ by M0 -- a 64-bit add on the ALU pipe instead of a multiply on the FMA-heavy pipe. */
__device__ __forceinline__ void zmc_philox_p0(zu64 p0, zu32 c1, zu32 c2, zu32 c3, const ZmcKeySchedule& ks, zu32* out) {
    zu32 c0;
    {
        const zu64 p1 = (zu64)c2 * (zu64)ZMC_PHILOX_M1;
        const zu32 n0 = (zu32)(p1 >> 32) ^ c1 ^ ks.k0[0];
        const zu32 n2 = (zu32)(p0 >> 32) ^ c3 ^ ks.k1[0];
        c1 = (zu32)p1;
        c3 = (zu32)p0;
        c0 = n0;
        c2 = n2;
    }
#pragma unroll
    for (int r = 1; r < 10; ++r) {
        const zu64 q0 = (zu64)c0 * (zu64)ZMC_PHILOX_M0;
        const zu64 q1 = (zu64)c2 * (zu64)ZMC_PHILOX_M1;
        const zu32 n0 = (zu32)(q1 >> 32) ^ c1 ^ ks.k0[r];
        const zu32 n2 = (zu32)(q0 >> 32) ^ c3 ^ ks.k1[r];
        c1 = (zu32)q1;
        c3 = (zu32)q0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R3: counter of call q of unit (path P, level l, trial t): (q, t | l<<8 | P[79:64]<<16, P[31:0], P[63:32]) */
struct ZmcUnitCounter {
    zu32 c1, c2, c3;
    __device__ __forceinline__ void init(zu64 path_lo, zu32 path_hi, zu32 level, zu32 trial) {
        c1 = trial | (level << 8) | ((path_hi & 0xFFFFu) << 16);
        c2 = (zu32)path_lo;
        c3 = (zu32)(path_lo >> 32);
    }
};

/* ------------------------------------------------------------------ R8: FP32 elementary functions (exact mode) */
/* zsin: k = rint(a/pi) by the magic-number add, two-constant Cody-Waite reduction, odd degree-9
 * polynomial on [-pi/2, pi/2], sign (-1)^k taken from the low bit of the magic sum. */
__device__ __forceinline__ float zmc_zsin(float a) {
    const float INV_PI = __uint_as_float(0x3ea2f983u);
    const float MAGIC = __uint_as_float(0x4b400000u);
    const float NPI_A = __uint_as_float(0xc0490000u);   /* -3.140625 */
    const float NPI_B = __uint_as_float(0xba7daa22u);   /* -fl(pi - 3.140625) */
    const float C3 = __uint_as_float(0xbe2aaaa6u), C5 = __uint_as_float(0x3c08876au);
    const float C7 = __uint_as_float(0xb94fb7f7u), C9 = __uint_as_float(0x362ede75u);
    const float t = __fmaf_rn(a, INV_PI, MAGIC);
    const float kf = __fadd_rn(t, -MAGIC);
    float r = __fmaf_rn(kf, NPI_A, a);
    r = __fmaf_rn(kf, NPI_B, r);
    const float s = __fmul_rn(r, r);
    float p = __fmaf_rn(C9, s, C7);
    p = __fmaf_rn(p, s, C5);
    p = __fmaf_rn(p, s, C3);
    const float rs = __fmul_rn(r, s);
    const float v = __fmaf_rn(rs, p, r);
    /* sign (-1)^k: bit 0 of t into bit 31 of v. v + (t << 31) mod 2^32 = v ^ ((t & 1) << 31): one IMAD */
    return __uint_as_float(__float_as_uint(t) * 0x80000000u + __float_as_uint(v));
}

/* zexp: n = rint(e*log2 e) by the magic-number add, two-constant reduction r = e - n ln2, degree-6
 * polynomial p ~ exp(r); exp(e) = p * 2^n is assembled as an FP64 number by adding n to the
 * exponent field of (double)p, so the FP64 exponent range is available (R9: the 9-D Gaussian's
 * samples at level 1 lie far below FP32's range). |e| > 708 and NaN take the slow branch. */
/* CHK = false: the caller has proved |e| <= 708 for every sample of the work item (ZmcIntegrand::setup, "range proof"),
 * so the test, its branch and the special values are not in the loop at all; the arithmetic is the same. */
template <bool CHK = true>
__device__ __forceinline__ double zmc_zexp_value(float e) {
    if (CHK && !(fabsf(e) <= 708.0f)) {
        if (e < 0.0f) return 0.0;
        if (e > 0.0f) return __longlong_as_double(0x7FF0000000000000ll);
        return __longlong_as_double(0x7FF8000000000000ll);
    }
    const float LOG2E = __uint_as_float(0x3fb8aa3bu);
    const float MAGIC = __uint_as_float(0x4b400000u);
    const float NLN2_HI = __uint_as_float(0xbf317200u);
    const float NLN2_LO = __uint_as_float(0xb5bfbe8eu);
    const float E2 = __uint_as_float(0x3efffffeu), E3 = __uint_as_float(0x3e2aaa49u), E4 = __uint_as_float(0x3d2aac79u);
    const float E5 = __uint_as_float(0x3c091cf1u), E6 = __uint_as_float(0x3ab5121au);
    const float t = __fmaf_rn(e, LOG2E, MAGIC);
    const float nf = __fadd_rn(t, -MAGIC);
    float r = __fmaf_rn(nf, NLN2_HI, e);
    r = __fmaf_rn(nf, NLN2_LO, r);
    float p = __fmaf_rn(E6, r, E5);
    p = __fmaf_rn(p, r, E4);
    p = __fmaf_rn(p, r, E3);
    p = __fmaf_rn(p, r, E2);
    p = __fmaf_rn(p, r, 1.0f);
    p = __fmaf_rn(p, r, 1.0f);
    /* n = bits(t) - 0x4b400000; only the low 12 bits of n survive "<< 20" and 0x4b400000 has none set,
     * so bits(t) << 20 is n << 20 */
    const double dp = (double)p;
    return __hiloint2double(__double2hiint(dp) + (zi32)(__float_as_uint(t) << 20), __double2loint(dp));
}

/* fast mode: the same split e*log2e = n + r, with 2^r from MUFU.EX2 */
template <bool CHK = true>
__device__ __forceinline__ double zmc_fexp_value(float e) {
    if (CHK && !(fabsf(e) <= 708.0f)) {
        if (e < 0.0f) return 0.0;
        if (e > 0.0f) return __longlong_as_double(0x7FF0000000000000ll);
        return __longlong_as_double(0x7FF8000000000000ll);
    }
    const float MAGIC = __uint_as_float(0x4b400000u);
    const float y = __fmul_rn(e, __uint_as_float(0x3fb8aa3bu));
    const float t = __fadd_rn(y, MAGIC);
    const float nf = __fadd_rn(t, -MAGIC);
    const float r = __fadd_rn(y, -nf);
    float p;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(p) : "f"(r));
    const zi32 n = (zi32)(__float_as_uint(t) - 0x4b400000u);
    const double dp = (double)p;
    return __hiloint2double(__double2hiint(dp) + (n << 20), __double2loint(dp));
}


/* ------------------------------------------------------------------ packed FP32 pairs (FFMA2 / FADD2 / FMUL2, new on sm_100) */
/* Two samples share one instruction: fma/add/mul.rn.f32x2 are component-wise IEEE round-to-nearest,
 * so a packed sequence gives bit for bit what the scalar sequence gives on each component (R8).
 * A broadcast operand (v, v) costs no register: ptxas encodes it as a scalar/immediate operand.
 * Why it pays: the path is bound by dispatch slots, and one FFMA2 costs less
 * than two FFMA there. */
typedef unsigned long long zf2;
__device__ __forceinline__ zf2 zmc_pk(float lo, float hi) { zf2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ zf2 zmc_bc(float v) { return zmc_pk(v, v); }
__device__ __forceinline__ float zmc_lo(zf2 v) { float a, b; asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); (void)b; return a; }
__device__ __forceinline__ float zmc_hi(zf2 v) { float a, b; asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); (void)a; return b; }
__device__ __forceinline__ zf2 zmc_fma2(zf2 a, zf2 b, zf2 c) { zf2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ zf2 zmc_add2(zf2 a, zf2 b) { zf2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ zf2 zmc_mul2(zf2 a, zf2 b) { zf2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

/* zmc_zsin on a pair: the same operation sequence, component-wise */
__device__ __forceinline__ zf2 zmc_zsin2(zf2 a) {
    const float INV_PI = __uint_as_float(0x3ea2f983u);
    const float MAGIC = __uint_as_float(0x4b400000u);
    const float NPI_A = __uint_as_float(0xc0490000u);
    const float NPI_B = __uint_as_float(0xba7daa22u);
    const float C3 = __uint_as_float(0xbe2aaaa6u), C5 = __uint_as_float(0x3c08876au);
    const float C7 = __uint_as_float(0xb94fb7f7u), C9 = __uint_as_float(0x362ede75u);
    const zf2 t = zmc_fma2(a, zmc_bc(INV_PI), zmc_bc(MAGIC));
    const zf2 kf = zmc_add2(t, zmc_bc(-MAGIC));
    zf2 r = zmc_fma2(kf, zmc_bc(NPI_A), a);
    r = zmc_fma2(kf, zmc_bc(NPI_B), r);
    const zf2 s = zmc_mul2(r, r);
    zf2 p = zmc_fma2(zmc_bc(C9), s, zmc_bc(C7));
    p = zmc_fma2(p, s, zmc_bc(C5));
    p = zmc_fma2(p, s, zmc_bc(C3));
    const zf2 rs = zmc_mul2(r, s);
    const zf2 v = zmc_fma2(rs, p, r);
    const zu32 vl = __float_as_uint(zmc_lo(t)) * 0x80000000u + __float_as_uint(zmc_lo(v));
    const zu32 vh = __float_as_uint(zmc_hi(t)) * 0x80000000u + __float_as_uint(zmc_hi(v));
    return zmc_pk(__uint_as_float(vl), __uint_as_float(vh));
}

/* zmc_zexp_value on a pair: packed reduction and polynomial, then each component assembled as there */
template <bool CHK>
__device__ __forceinline__ double zmc_zexp_finish(float e, float t, float p) {
    const double dp = (double)p;
    double v = __hiloint2double(__double2hiint(dp) + (zi32)(__float_as_uint(t) << 20), __double2loint(dp));
    if (CHK && !(fabsf(e) <= 708.0f))
        v = (e < 0.0f) ? 0.0 : ((e > 0.0f) ? __longlong_as_double(0x7FF0000000000000ll) : __longlong_as_double(0x7FF8000000000000ll));
    return v;
}
template <bool CHK>
__device__ __forceinline__ void zmc_zexp2(zf2 e, double& fa, double& fb) {
    const float LOG2E = __uint_as_float(0x3fb8aa3bu);
    const float MAGIC = __uint_as_float(0x4b400000u);
    const float NLN2_HI = __uint_as_float(0xbf317200u);
    const float NLN2_LO = __uint_as_float(0xb5bfbe8eu);
    const float E2 = __uint_as_float(0x3efffffeu), E3 = __uint_as_float(0x3e2aaa49u), E4 = __uint_as_float(0x3d2aac79u);
    const float E5 = __uint_as_float(0x3c091cf1u), E6 = __uint_as_float(0x3ab5121au);
    const zf2 t = zmc_fma2(e, zmc_bc(LOG2E), zmc_bc(MAGIC));
    const zf2 nf = zmc_add2(t, zmc_bc(-MAGIC));
    zf2 r = zmc_fma2(nf, zmc_bc(NLN2_HI), e);
    r = zmc_fma2(nf, zmc_bc(NLN2_LO), r);
    zf2 p = zmc_fma2(zmc_bc(E6), r, zmc_bc(E5));
    p = zmc_fma2(p, r, zmc_bc(E4));
    p = zmc_fma2(p, r, zmc_bc(E3));
    p = zmc_fma2(p, r, zmc_bc(E2));
    p = zmc_fma2(p, r, zmc_bc(1.0f));
    p = zmc_fma2(p, r, zmc_bc(1.0f));
    fa = zmc_zexp_finish<CHK>(zmc_lo(e), zmc_lo(t), zmc_lo(p));
    fb = zmc_zexp_finish<CHK>(zmc_hi(e), zmc_hi(t), zmc_hi(p));
}

/* ------------------------------------------------------------------ R2 + R4: cell geometry and the word -> point map */
/* lo_d = lower_d + (double)I_d * width_d (multiply, then add).
 * FP64: x = lo + ((double)w + 0.5) * (width * 2^-32).
 * FP32: u' = bits(0x3F800000 | w>>9) in [1,2) ; x = fmaf(u', (float)width, base),
 *       base = (float)(((lo - width) + width*2^-24) - centre), formed in FP64. */
template <int D>
struct ZmcMapF32 {
    float wf[D], base[D];
    __device__ __forceinline__ void init_dim(int d, double lower, double width, zu32 coord, double centre) {
        const double lo = __dadd_rn(lower, __dmul_rn((double)coord, width));
        double b = __dadd_rn(__dadd_rn(lo, -width), __dmul_rn(width, 5.9604644775390625e-08));
        b = __dadd_rn(b, -centre);
        base[d] = (float)b;
        wf[d] = (float)width;
    }
    __device__ __forceinline__ float x(int d, zu32 w) const {
        return __fmaf_rn(__uint_as_float(0x3F800000u | (w >> 9)), wf[d], base[d]);
    }
    __device__ __forceinline__ zf2 x2(int d, zu32 wa, zu32 wb) const {   /* two samples' coordinate d */
        return zmc_fma2(zmc_pk(__uint_as_float(0x3F800000u | (wa >> 9)), __uint_as_float(0x3F800000u | (wb >> 9))),
                        zmc_bc(wf[d]), zmc_bc(base[d]));
    }
};

/* ------------------------------------------------------------------ FP64 sine (R8: FP64 values within 4 ulp of the CPU's libm) */
/* The FP32 scheme at FP64 length, branch-free: k = rint(a/pi) by the magic-number add, three-constant Cody-Waite reduction with FMAs
 * (a - k*PI_HI is exact: a multiple of 2^-51 below 1.6), odd polynomial of degree 17 on [-pi/2, pi/2] (near-minimax: interpolation of
 * (sin(r)/r - 1)/r^2 at 8 Chebyshev nodes in r^2), sign (-1)^k from the low bit of the magic sum. 15 FP64 instructions against ~28 of
 * libdevice's sin with its quadrant selection, and no call. Measured against sinl on the host with the same operations (gcc, fma()):
 * at most 1.94 ulp for |a| <= 1e9 (the worst cases sit at |r| near pi/2, where r + r^3 p cancels 1.57 - 0.57), 0.99 ulp at a = fl(k pi);
 * libm itself is within 0.52, so the two sides differ by at most 2.5 ulp. Beyond 2^30 (k*PI_LO's own error starts to show in r):
 * libdevice's sin, with its Payne-Hanek reduction. */
static __device__ __noinline__ double zmc_sin_far(double a) { return sin(a); }      /* one cold copy per program, called: not inlined into every sample loop */

__device__ __forceinline__ double zmc_zsin64(double a) {
    if (!(fabs(a) <= 1073741824.0)) return zmc_sin_far(a);      /* also NaN and infinity */
    const double MAGIC = 6755399441055744.0;            /* 1.5 * 2^52: adding it rounds to an integer in the low mantissa bits */
    const double t = __fma_rn(a, __longlong_as_double(0x3fd45f306dc9c883ll), MAGIC);       /* a/pi + MAGIC */
    const double kd = __dadd_rn(t, -MAGIC);
    double r = __fma_rn(-kd, __longlong_as_double(0x400921fb54442d18ll), a);                /* PI_HI */
    r = __fma_rn(-kd, __longlong_as_double(0x3ca1a62633145c07ll), r);                        /* PI_MID */
    r = __fma_rn(-kd, __longlong_as_double(0xb92f1976b7ed8fbcll), r);                        /* PI_LO */
    const double r2 = __dmul_rn(r, r);
    double p = __longlong_as_double(0x3ce892efd890db97ll);                                   /* r^17 */
    p = __fma_rn(p, r2, __longlong_as_double(0xbd6ae4d771729416ll));
    p = __fma_rn(p, r2, __longlong_as_double(0x3de6123f55a16315ll));
    p = __fma_rn(p, r2, __longlong_as_double(0xbe5ae64557c0cbf9ll));
    p = __fma_rn(p, r2, __longlong_as_double(0x3ec71de3a5419df5ll));
    p = __fma_rn(p, r2, __longlong_as_double(0xbf2a01a01a0184f4ll));
    p = __fma_rn(p, r2, __longlong_as_double(0x3f81111111111104ll));
    p = __fma_rn(p, r2, __longlong_as_double(0xbfc5555555555555ll));                         /* r^3 */
    const double v = __fma_rn(__dmul_rn(r, r2), p, r);
    return __hiloint2double(__double2hiint(v) ^ (__double2loint(t) << 31), __double2loint(v));
}

template <int D>
struct ZmcMapF64 {
    double lo[D], step[D];
    __device__ __forceinline__ void init_dim(int d, double lower, double width, zu32 coord) {
        lo[d] = __dadd_rn(lower, __dmul_rn((double)coord, width));
        step[d] = __dmul_rn(width, 2.3283064365386963e-10);
    }
    __device__ __forceinline__ double x(int d, zu32 w) const {
        /* (double)w + 0.5 without the conversion: bits (0x43300000 : w) are the double 2^52 + w, and (2^52 + w) - (2^52 - 0.5) is
         * exact -- one DADD instead of I2F.F64.U32 (XU pipe, 8.5 clocks per warp-instruction) + DADD; the same value bit for bit */
        const double wh = __dadd_rn(__hiloint2double(0x43300000, (zi32)w), -4503599627370495.5);
        return __dadd_rn(lo[d], __dmul_rn(wh, step[d]));
    }
};

#ifndef ZMC_PACKED_SIN_POLY
#define ZMC_PACKED_SIN_POLY(D) 1
#endif
#ifndef ZMC_PACKED_EXP_POLY
#define ZMC_PACKED_EXP_POLY(D) ((D) <= 8)
#endif

/* two copies of the sample loop (with and without zexp's range test) pay where the polynomial is packed; with the scalar
 * polynomial of D >= 9 ptxas needs 50-60 more registers for them (measured) and most cells of a narrow Gaussian are out of range anyway */
#ifndef ZMC_RANGE_PROOF
#define ZMC_RANGE_PROOF(D) ZMC_PACKED_EXP_POLY(D)
#endif

/* ------------------------------------------------------------------ integrands */
/* Each integrand policy has
 *   setup(args, instance, coords)  once per work item: geometry and this instance's parameters
 *   eval(words, xout)              one sample from D consecutive words -> the FP64 value the unit sum adds
 *                                  (xout != nullptr only in the debug kernel). */
/* ZMC_USER_NC (R15): 0 = the user function returns its one value; n >= 1 = it is vector-valued and writes n components
 * f_0 .. f_{n-1} of the same point: one word stream, one map, n FP64 sums per (cell, trial) unit. */
#ifndef ZMC_USER_NC
#define ZMC_USER_NC 0
#endif
#define ZMC_DEV_MAX_COMPONENTS 16
#ifdef ZMC_USER_FN
#if ZMC_USER_NC > 0
__device__ void ZMC_USER_FN(const float* x, int dim, const float* p, int np, float* out, int n_out);
__device__ void ZMC_USER_FN(const double* x, int dim, const double* p, int np, double* out, int n_out);
#else
__device__ float ZMC_USER_FN(const float* x, int dim, const float* p, int np);
__device__ double ZMC_USER_FN(const double* x, int dim, const double* p, int np);
#endif
#endif
template <int ID> struct ZmcComponents {
    static constexpr bool VEC = (ID == ZMC_ID_USER) && (ZMC_USER_NC > 0);
    static constexpr int NC = VEC ? ZMC_USER_NC : 1;
};

template <int ID, int D_, int PREC, int MODE>
struct ZmcIntegrand;

template <int ID, int D_, int MODE>
struct ZmcIntegrand<ID, D_, ZMC_PREC_F32, MODE> {
    static constexpr int D = D_;
    static constexpr int PREC = ZMC_PREC_F32;
    static constexpr bool VEC = ZmcComponents<ID>::VEC;
    static constexpr int NC = ZmcComponents<ID>::NC;
    ZmcMapF32<D_> map;
    float c0;           /* CONST/LINEAR: p[0] ; EXP_QUAD: -a */
    float lin[ID == ZMC_ID_LINEAR ? D_ : 1];
    const float* up;    /* user parameters */
    zi32 unp;
    /* EXP_QUAD: true if |e| = |a|*q <= 708 is proved for every point of this cell, so that the sample loop can run
     * without the per-sample range test of zexp (same arithmetic, fewer instructions); false = test every sample */
    static constexpr bool HAS_RANGE_PROOF = (ID == ZMC_ID_EXP_QUAD) && ZMC_RANGE_PROOF(D_);
    bool in_range;

    __device__ __forceinline__ void setup(const ZmcSampleArgs& a, zu32 inst, const zu32* coords) {
        const double* p = a.params + (zu64)inst * (zu64)a.ppi;
#pragma unroll
        for (int d = 0; d < D_; ++d) {
            const double centre = (ID == ZMC_ID_EXP_QUAD) ? p[2 + d] : 0.0;
            map.init_dim(d, a.lower[d], a.width[d], coords[d], centre);
        }
        c0 = 0.0f;
        if (ID == ZMC_ID_CONST || ID == ZMC_ID_LINEAR) c0 = (float)p[0];
        if (ID == ZMC_ID_EXP_QUAD) c0 = -(float)p[1];
        if (ID == ZMC_ID_LINEAR) {
#pragma unroll
            for (int d = 0; d < D_; ++d) lin[d] = (float)p[1 + d];
        }
        up = a.params_f32 + (zu64)inst * (zu64)a.ppi;
        unp = a.ppi;
        in_range = false;
        if (HAS_RANGE_PROOF) {
            /* x_d = fmaf(u', wf, base) is monotone in u' in [1, 2): |x_d| <= max(|fl(wf+base)|, |fl(2wf+base)|) =: m_d.
             * q <= (sum m_d^2)(1 + D*2^-23) in FP32 ; the bound carries a 2^-7 margin and the limit 700 leaves 8 more */
            float qmax = 0.0f;
#pragma unroll
            for (int d = 0; d < D_; ++d) {
                const float xa = fabsf(__fmaf_rn(1.0f, map.wf[d], map.base[d]));
                const float xb = fabsf(__fmaf_rn(2.0f, map.wf[d], map.base[d]));
                const float md = fmaxf(xa, xb);
                qmax = __fmaf_rn(md, md, qmax);
            }
            in_range = __fmul_rn(__fmul_rn(fabsf(c0), qmax), 1.0078125f) <= 700.0f;      /* NaN: false */
        }
    }

    template <bool CHK = true>
    __device__ __forceinline__ double eval(const zu32* w, double* xout) const {
        float x[D_];
#pragma unroll
        for (int d = 0; d < D_; ++d) x[d] = map.x(d, w[d]);
        if (xout) {
#pragma unroll
            for (int d = 0; d < D_; ++d) xout[d] = (double)x[d];
        }
        if (ID == ZMC_ID_CONST) return (double)c0;
        if (ID == ZMC_ID_LINEAR) {
            float f = c0;
#pragma unroll
            for (int d = 0; d < D_; ++d) f = __fmaf_rn(lin[d], x[d], f);
            return (double)f;
        }
        if (ID == ZMC_ID_SIN_SUM) {          /* paper f1, Eq. (1) */
            float s = x[0];
#pragma unroll
            for (int d = 1; d < D_; ++d) s = __fadd_rn(s, x[d]);
            if (MODE == ZMC_MODE_FAST) return (double)__sinf(s);
            return (double)zmc_zsin(s);
        }
        if (ID == ZMC_ID_EXP_QUAD) {         /* paper f2, Eq. (2); x holds x - c */
            float q = __fmul_rn(x[0], x[0]);
#pragma unroll
            for (int d = 1; d < D_; ++d) q = __fmaf_rn(x[d], x[d], q);
            const float e = __fmul_rn(c0, q);
            if (MODE == ZMC_MODE_FAST) return zmc_fexp_value<CHK>(e);
            return zmc_zexp_value<CHK>(e);
        }
#if defined(ZMC_USER_FN) && ZMC_USER_NC == 0
        if (ID == ZMC_ID_USER) return (double)ZMC_USER_FN((const float*)x, D_, up, unp);
#endif
        return 0.0;
    }

    /* R15: the NC components of a vector-valued user integrand at one sample point */
    __device__ __forceinline__ void evalv(const zu32* w, double* out, double* xout) const {
        float x[D_];
#pragma unroll
        for (int d = 0; d < D_; ++d) x[d] = map.x(d, w[d]);
        if (xout) {
#pragma unroll
            for (int d = 0; d < D_; ++d) xout[d] = (double)x[d];
        }
#if defined(ZMC_USER_FN) && ZMC_USER_NC > 0
        float o[NC];
        ZMC_USER_FN((const float*)x, D_, up, unp, o, NC);
#pragma unroll
        for (int j = 0; j < NC; ++j) out[j] = (double)o[j];
#else
        out[0] = eval(w, nullptr);
#endif
    }

    /* Two samples at once on the packed FP32 instructions: component-wise the operation sequence of eval(),
     * hence the same bits (checked by the P1 parity test through zmc_points_kernel). */
    static constexpr bool HAS_PACKED = (ID == ZMC_ID_SIN_SUM || ID == ZMC_ID_EXP_QUAD || ID == ZMC_ID_LINEAR);
    template <bool CHK = true>
    __device__ __forceinline__ void eval2(const zu32* wa, const zu32* wb, double& fa, double& fb) const {
        if (!HAS_PACKED) { fa = eval<CHK>(wa, nullptr); fb = eval<CHK>(wb, nullptr); return; }
        zf2 x[D_];
#pragma unroll
        for (int d = 0; d < D_; ++d) x[d] = map.x2(d, wa[d], wb[d]);
        if (ID == ZMC_ID_LINEAR) {
            zf2 f = zmc_bc(c0);
#pragma unroll
            for (int d = 0; d < D_; ++d) f = zmc_fma2(zmc_bc(lin[d]), x[d], f);
            fa = (double)zmc_lo(f);
            fb = (double)zmc_hi(f);
        }
        if (ID == ZMC_ID_SIN_SUM) {
            zf2 s = x[0];
#pragma unroll
            for (int d = 1; d < D_; ++d) s = zmc_add2(s, x[d]);
            if (MODE == ZMC_MODE_FAST) {
                fa = (double)__sinf(zmc_lo(s));
                fb = (double)__sinf(zmc_hi(s));
            } else if (ZMC_PACKED_SIN_POLY(D_)) {
                const zf2 v = zmc_zsin2(s);
                fa = (double)zmc_lo(v);
                fb = (double)zmc_hi(v);
            } else {
                fa = (double)zmc_zsin(zmc_lo(s));
                fb = (double)zmc_zsin(zmc_hi(s));
            }
        }
        if (ID == ZMC_ID_EXP_QUAD) {
            zf2 q = zmc_mul2(x[0], x[0]);
#pragma unroll
            for (int d = 1; d < D_; ++d) q = zmc_fma2(x[d], x[d], q);
            const zf2 e = zmc_mul2(zmc_bc(c0), q);
            if (MODE == ZMC_MODE_FAST) {
                fa = zmc_fexp_value<CHK>(zmc_lo(e));
                fb = zmc_fexp_value<CHK>(zmc_hi(e));
            } else if (ZMC_PACKED_EXP_POLY(D_)) {
                zmc_zexp2<CHK>(e, fa, fb);
            } else {      /* packed map and quadratic form, scalar polynomial: fewer live registers at high D */
                fa = zmc_zexp_value<CHK>(zmc_lo(e));
                fb = zmc_zexp_value<CHK>(zmc_hi(e));
            }
        }
    }
};

template <int ID, int D_, int MODE>
struct ZmcIntegrand<ID, D_, ZMC_PREC_F64, MODE> {
    static constexpr int D = D_;
    static constexpr int PREC = ZMC_PREC_F64;
    static constexpr bool VEC = ZmcComponents<ID>::VEC;
    static constexpr int NC = ZmcComponents<ID>::NC;
    ZmcMapF64<D_> map;
    double c0;          /* CONST/LINEAR: p[0] ; EXP_QUAD: a */
    double aux[(ID == ZMC_ID_LINEAR || ID == ZMC_ID_EXP_QUAD) ? D_ : 1];   /* LINEAR: coefficients ; EXP_QUAD: centre */
    const double* up;
    zi32 unp;

    __device__ __forceinline__ void setup(const ZmcSampleArgs& a, zu32 inst, const zu32* coords) {
        const double* p = a.params + (zu64)inst * (zu64)a.ppi;
#pragma unroll
        for (int d = 0; d < D_; ++d) map.init_dim(d, a.lower[d], a.width[d], coords[d]);
        c0 = 0.0;
        if (ID == ZMC_ID_CONST || ID == ZMC_ID_LINEAR) c0 = p[0];
        if (ID == ZMC_ID_EXP_QUAD) c0 = p[1];
        if (ID == ZMC_ID_LINEAR) {
#pragma unroll
            for (int d = 0; d < D_; ++d) aux[d] = p[1 + d];
        }
        if (ID == ZMC_ID_EXP_QUAD) {
#pragma unroll
            for (int d = 0; d < D_; ++d) aux[d] = p[2 + d];
        }
        up = p;
        unp = a.ppi;
    }

    static constexpr bool HAS_RANGE_PROOF = false;
    static constexpr bool in_range = false;
    template <bool CHK = true>
    __device__ __forceinline__ double eval(const zu32* w, double* xout) const {
        double x[D_];
#pragma unroll
        for (int d = 0; d < D_; ++d) x[d] = map.x(d, w[d]);
        if (xout) {
#pragma unroll
            for (int d = 0; d < D_; ++d) xout[d] = x[d];
        }
        if (ID == ZMC_ID_CONST) return c0;
        if (ID == ZMC_ID_LINEAR) {
            double f = c0;
#pragma unroll
            for (int d = 0; d < D_; ++d) f = __dadd_rn(f, __dmul_rn(aux[d], x[d]));
            return f;
        }
        if (ID == ZMC_ID_SIN_SUM) {
            double s = x[0];
#pragma unroll
            for (int d = 1; d < D_; ++d) s = __dadd_rn(s, x[d]);
            return zmc_zsin64(s);
        }
        if (ID == ZMC_ID_EXP_QUAD) {
            double q = 0.0;
#pragma unroll
            for (int d = 0; d < D_; ++d) {
                const double y = __dadd_rn(x[d], -aux[d]);
                const double yy = __dmul_rn(y, y);
                q = (d == 0) ? yy : __dadd_rn(q, yy);
            }
            return exp(-__dmul_rn(c0, q));
        }
#if defined(ZMC_USER_FN) && ZMC_USER_NC == 0
        if (ID == ZMC_ID_USER) return ZMC_USER_FN((const double*)x, D_, up, unp);
#endif
        return 0.0;
    }
    __device__ __forceinline__ void evalv(const zu32* w, double* out, double* xout) const {
        double x[D_];
#pragma unroll
        for (int d = 0; d < D_; ++d) x[d] = map.x(d, w[d]);
        if (xout) {
#pragma unroll
            for (int d = 0; d < D_; ++d) xout[d] = x[d];
        }
#if defined(ZMC_USER_FN) && ZMC_USER_NC > 0
        ZMC_USER_FN((const double*)x, D_, up, unp, out, NC);
#else
        out[0] = eval(w, nullptr);
#endif
    }
    static constexpr bool HAS_PACKED = false;   /* there is no packed FP64 */
    template <bool CHK = true>
    __device__ __forceinline__ void eval2(const zu32* wa, const zu32* wb, double& fa, double& fb) const {
        fa = eval<CHK>(wa, nullptr);
        fb = eval<CHK>(wb, nullptr);
    }
};

/* ------------------------------------------------------------------ work-item decoding (R2) */
/* item -> (cell, trial, chunk); cell -> (parent G, child j); child j -> digits j_d (axis 0 least
 * significant), I'_d = I_d*g + j_d ; path P' = P*k + j (80 bits). */
/* n = q*d + r. Work-item indices and child indices are below 2^32 except on the very largest levels: the 32-bit division is
 * ~15 inline instructions, the 64-bit one a subroutine call of ~100 -- and there are 3 + D of them per work item. */
template <bool FAST>
__device__ __forceinline__ void zmc_divmod(zu64 n, zu32 d, zu64& q, zu32& r) {
    if (FAST && (n >> 32) == 0ull) {
        const zu32 q32 = (zu32)n / d;
        r = (zu32)n - q32 * d;
        q = q32;
    } else {
        const zu64 q64 = n / d;
        r = (zu32)(n - q64 * d);
        q = q64;
    }
}

template <int D>
struct ZmcUnit {
    zu32 inst, trial, chunk;
    zu64 cell;
    zu64 path_lo;
    zu32 path_hi;
    zu32 coords[D];
    template <bool FAST>
    __device__ __forceinline__ void decode(const ZmcSampleArgs& a, zu64 item, zu32 n_chunks, zu32 trials_per_item) {
        zu64 unit;
        zmc_divmod<FAST>(item, n_chunks, unit, chunk);
        if (trials_per_item == 1u) zmc_divmod<FAST>(unit, a.T, cell, trial);
        else { cell = unit; trial = 0u; }       /* the item is the whole cell: trials 0 .. T-1 */
        zu64 G, j;
        if (FAST && ((cell | a.k) >> 32) == 0ull) {     /* the usual case, without the 64-bit division routine */
            const zu32 G32 = (zu32)cell / (zu32)a.k;
            G = G32;
            j = (zu32)cell - G32 * (zu32)a.k;
        } else {
            G = cell / a.k;
            j = cell - G * a.k;
        }
        inst = a.par_inst[G];
        const zu64 plo = a.par_plo[G];
        const zu32 phi = a.par_phi[G];
        path_lo = plo * a.k + j;
        const zu64 carry = __umul64hi(plo, a.k) + ((path_lo < j) ? 1ull : 0ull);
        path_hi = (zu32)((zu64)phi * a.k + carry);
#pragma unroll
        for (int d = 0; d < D; ++d) {
            zu32 jd;
            zmc_divmod<FAST>(j, a.g, j, jd);
            coords[d] = a.par_coord[(zu64)d * a.par_stride + G] * a.g + jd;
        }
    }
};

/* ------------------------------------------------------------------ the fused sampling kernel */
/* Flat word stream (R3): sample s, dimension d uses word s*D + d of the unit's stream; word i lives
 * in Philox call i>>2, lane i&3. A "group" is the smallest run of samples that starts on a call
 * boundary: SG = 4/gcd(D,4) samples = CG = D/gcd(D,4) calls. */
template <int D> struct ZmcGroup {
    static constexpr int G4 = (D % 4 == 0) ? 4 : ((D % 2 == 0) ? 2 : 1);
    static constexpr int SG = 4 / G4;
    static constexpr int CG = D / G4;
};

/* Per-instance tuning of the sampling kernel (measured on B200; profiles/r1_variants.md). The path is
 * bound by dispatch slots, so what is tuned is the instruction count and the compiler's schedule:
 *   PACKED  evaluate two samples per FFMA2/FADD2/FMUL2 (needs F::HAS_PACKED)
 *   UNROLL  sample groups in flight per lane and loop trip: 2 or 4
 *   MINB    resident CTAs per SM asked of __launch_bounds__ (register cap)
 *   P0_ADD  first-round products M0*q of a group's later calls by 64-bit addition (ALU pipe) instead of IMAD.WIDE
 *   P0_CARRY  ... and the group's own first product as a 64-bit induction variable of the sample loop:
 *           no first-round multiply at all on the FMA-heavy pipe
 *   FAST_DECODE  32-bit divisions in the item decoding where the operands allow (neutral in time, fewer instructions)
 *   TRIAL_LOOP   the kernel honours ZmcLevelInfo::trials_per_item (one item = all T trials of a cell; decoding, geometry and the
 *           latency chain atomic -> parent record -> key/parameters once per cell): +3 % at D = 4, N = 4096; +4.6 % at D = 3,
 *           N = 2000; +1 % at D = 12; nothing at N >= 1e5. Off: every item is one (cell, trial, chunk) unit
 *           (profiles/r2_variants.md) */
/* which kernels loop over the trials of a cell (TRIAL_LOOP below); the host asks too: it plans trials_per_item accordingly.
 * At D = 6 the loop costs 30 registers (118 -> 148: 3 CTAs per SM instead of 4) and 2 % at N = 1e5. */
__host__ __device__ constexpr bool zmc_tune_trial_loop(int D) { return D != 6; }

template <class F>
struct ZmcTune {
    static constexpr int D = F::D;
    static constexpr bool PACKED = F::HAS_PACKED;
    static constexpr int UNROLL = (D == 4 || D == 6 || D == 12) ? 4 : 2;
    static constexpr bool P0_ADD = (D == 4 || D == 6 || D == 12);   /* +3.7 % at D = 6, +1 % at D = 4 and 12, -1.5 % at D = 9 */
    static constexpr bool P0_CARRY = P0_ADD;
    /* FP64: at high D the kernel spills below 255 registers (2 CTAs; the 9-D Gaussian keeps 16 bytes of spill even there); the FP64 6-D kernel is
     * latency-bound and gains from a fifth CTA per SM (90 registers instead of 104: 0.551 -> 0.567 of the roof, profiles/r3_fp64_pipe_split.md) */
    static constexpr int MINB = (F::PREC == ZMC_PREC_F64) ? (D >= 7 ? 2 : (D == 6 ? 4 : 3)) : 3;
    static constexpr bool FAST_DECODE = true;
    static constexpr bool TRIAL_LOOP = zmc_tune_trial_loop(D);
};

/* R13: q + f*f. FP32-mode values have 24 significant bits, so the product is exact and one DFMA is the
 * rounded-product-then-add of the definition; FP64 values get the two operations. */
template <class F>
__device__ __forceinline__ double zmc_sq_add(double q, double f) {
    return (F::PREC == ZMC_PREC_F32) ? __fma_rn(f, f, q) : __dadd_rn(q, __dmul_rn(f, f));
}

template <class F, bool SQ, bool CHK = true>
__device__ __forceinline__ void zmc_group_eval(const F& f, const ZmcKeySchedule& ks, const ZmcUnitCounter& uc, zu32 gi,
                                               double* acc, double* accq, zu64 pg = 0ull, bool have_pg = false) {
    constexpr int D = F::D, SG = ZmcGroup<D>::SG, CG = ZmcGroup<D>::CG;
    zu32 w[4 * CG];
    const zu32 q0 = gi * (zu32)CG;
    if (ZmcTune<F>::P0_ADD) {      /* one first-round multiply per group, the other calls' products by adding M0 */
        const zu64 p0 = have_pg ? pg : (zu64)q0 * (zu64)ZMC_PHILOX_M0;
#pragma unroll
        for (int c = 0; c < CG; ++c) zmc_philox_p0(p0 + (zu64)c * (zu64)ZMC_PHILOX_M0, uc.c1, uc.c2, uc.c3, ks, &w[4 * c]);
    } else {
#pragma unroll
        for (int c = 0; c < CG; ++c) zmc_philox(q0 + (zu32)c, uc.c1, uc.c2, uc.c3, ks, &w[4 * c]);
    }
    if (ZmcTune<F>::PACKED && SG >= 2) {      /* samples (2i, 2i+1) of the group as one packed evaluation */
#pragma unroll
        for (int s = 0; s < SG; s += 2) {
            double fa, fb;
            f.template eval2<CHK>(&w[s * D], &w[(s + 1) * D], fa, fb);
            acc[s] = __dadd_rn(acc[s], fa);
            acc[s + 1] = __dadd_rn(acc[s + 1], fb);
            if (SQ) { accq[0] = zmc_sq_add<F>(accq[0], fa); accq[1] = zmc_sq_add<F>(accq[1], fb); }
        }
    } else {
#pragma unroll
        for (int s = 0; s < SG; ++s) {
            const double fv = f.template eval<CHK>(&w[s * D], nullptr);
            acc[s] = __dadd_rn(acc[s], fv);
            if (SQ) accq[s & 1] = zmc_sq_add<F>(accq[s & 1], fv);
        }
    }
}

/* groups gi and gj: acc[0..SG) takes gi's samples, acc[SG..2SG) gj's -- the same sums as two zmc_group_eval calls */
template <class F, bool SQ, bool CHK = true>
__device__ __forceinline__ void zmc_group_eval_pair(const F& f, const ZmcKeySchedule& ks, const ZmcUnitCounter& uc, zu32 gi,
                                                    zu32 gj, double* acc, double* accq, zu64 pg = 0ull, bool have_pg = false) {
    constexpr int D = F::D, SG = ZmcGroup<D>::SG, CG = ZmcGroup<D>::CG;
    if (ZmcTune<F>::PACKED && SG == 1) {      /* one sample per group (D = 4, 8, ..): pack across the two groups */
        zu32 wa[4 * CG], wb[4 * CG];
        if (ZmcTune<F>::P0_ADD) {
            const zu64 pa = have_pg ? pg : (zu64)(gi * (zu32)CG) * (zu64)ZMC_PHILOX_M0;
            const zu64 pb = have_pg ? pg + (zu64)(32 * CG) * (zu64)ZMC_PHILOX_M0 : (zu64)(gj * (zu32)CG) * (zu64)ZMC_PHILOX_M0;
#pragma unroll
            for (int c = 0; c < CG; ++c) zmc_philox_p0(pa + (zu64)c * (zu64)ZMC_PHILOX_M0, uc.c1, uc.c2, uc.c3, ks, &wa[4 * c]);
#pragma unroll
            for (int c = 0; c < CG; ++c) zmc_philox_p0(pb + (zu64)c * (zu64)ZMC_PHILOX_M0, uc.c1, uc.c2, uc.c3, ks, &wb[4 * c]);
        } else {
#pragma unroll
            for (int c = 0; c < CG; ++c) zmc_philox(gi * (zu32)CG + (zu32)c, uc.c1, uc.c2, uc.c3, ks, &wa[4 * c]);
#pragma unroll
            for (int c = 0; c < CG; ++c) zmc_philox(gj * (zu32)CG + (zu32)c, uc.c1, uc.c2, uc.c3, ks, &wb[4 * c]);
        }
        double fa, fb;
        f.template eval2<CHK>(wa, wb, fa, fb);
        acc[0] = __dadd_rn(acc[0], fa);
        acc[1] = __dadd_rn(acc[1], fb);
        if (SQ) { accq[0] = zmc_sq_add<F>(accq[0], fa); accq[1] = zmc_sq_add<F>(accq[1], fb); }
    } else {
        /* gj = gi + 32: its first product is gi's plus 32*CG*M0 */
        zmc_group_eval<F, SQ, CHK>(f, ks, uc, gi, acc, accq, pg, have_pg);
        zmc_group_eval<F, SQ, CHK>(f, ks, uc, gj, acc + SG, accq + 2, pg + (zu64)(32 * CG) * (zu64)ZMC_PHILOX_M0, have_pg);
    }
}

/* One lane's share of a work item: the full sample groups gi, gi + 32, ... < gfe. acc[0..SG) sums the groups at even
 * multiples of 32 from the lane's first one, acc[SG..2SG) those at odd multiples -- whatever UNROLL is. */
template <class F, bool SQ, bool CHK>
__device__ __forceinline__ void zmc_full_groups(const F& f, const ZmcKeySchedule& ks, const ZmcUnitCounter& uc, zu32 gi, zu32 gfe,
                                                double* acc, double* accq) {
    constexpr int CG = ZmcGroup<F::D>::CG;
    constexpr bool CARRY = ZmcTune<F>::P0_CARRY;     /* the group's first product as a 64-bit induction variable */
    zu64 pg = (zu64)(gi * (zu32)CG) * (zu64)ZMC_PHILOX_M0;
    if (ZmcTune<F>::UNROLL == 8) {
        for (; gi + 224u < gfe; gi += 256u) {
#pragma unroll
            for (int h = 0; h < 4; ++h)
                zmc_group_eval_pair<F, SQ, CHK>(f, ks, uc, gi + 64u * h, gi + 64u * h + 32u, acc, accq, pg + (zu64)(64 * h * CG) * (zu64)ZMC_PHILOX_M0, CARRY);
            pg += (zu64)(256 * CG) * (zu64)ZMC_PHILOX_M0;
        }
    }
    if (ZmcTune<F>::UNROLL >= 4) {
        for (; gi + 96u < gfe; gi += 128u) {
            zmc_group_eval_pair<F, SQ, CHK>(f, ks, uc, gi, gi + 32u, acc, accq, pg, CARRY);
            zmc_group_eval_pair<F, SQ, CHK>(f, ks, uc, gi + 64u, gi + 96u, acc, accq, pg + (zu64)(64 * CG) * (zu64)ZMC_PHILOX_M0, CARRY);
            pg += (zu64)(128 * CG) * (zu64)ZMC_PHILOX_M0;
        }
    }
    for (; gi + 32u < gfe; gi += 64u) {
        zmc_group_eval_pair<F, SQ, CHK>(f, ks, uc, gi, gi + 32u, acc, accq, pg, CARRY);
        pg += (zu64)(64 * CG) * (zu64)ZMC_PHILOX_M0;
    }
    if (gi < gfe) zmc_group_eval<F, SQ, CHK>(f, ks, uc, gi, acc, accq);
}

/* R15: one unit of a vector-valued integrand -- the same word stream and the same points as a scalar unit, NC FP64 sums,
 * stored component-fastest at partial[out * NC + j]. One accumulator per component and lane (the user function, not the
 * generator, sets the pace here), plain Philox calls. */
template <class F, bool SQ>
__device__ __forceinline__ void zmc_unit_vec(const ZmcSampleArgs& a, const F& f, const ZmcKeySchedule& ks, const ZmcUnitCounter& uc,
                                             zu32 lane, zu32 gb, zu32 ge, zu32 gfe, zu32 full_groups, zu32 tail, zu64 out) {
    constexpr int D = F::D, SG = ZmcGroup<D>::SG, CG = ZmcGroup<D>::CG, NC = F::NC;
    double acc[NC], accq[SQ ? NC : 1];      /* SQ (R13 per component): sums of f_j^2 as well */
#pragma unroll
    for (int j = 0; j < NC; ++j) acc[j] = 0.0;
    if (SQ) {
#pragma unroll
        for (int j = 0; j < (SQ ? NC : 1); ++j) accq[j] = 0.0;
    }
    for (zu32 gi = gb + lane; gi < gfe; gi += 32u) {
        zu32 w[4 * CG];
#pragma unroll
        for (int c = 0; c < CG; ++c) zmc_philox(gi * (zu32)CG + (zu32)c, uc.c1, uc.c2, uc.c3, ks, &w[4 * c]);
#pragma unroll
        for (int s = 0; s < SG; ++s) {
            double o[NC];
            f.evalv(&w[s * D], o, nullptr);
#pragma unroll
            for (int j = 0; j < NC; ++j) acc[j] = __dadd_rn(acc[j], o[j]);
            if (SQ) {
#pragma unroll
                for (int j = 0; j < (SQ ? NC : 1); ++j) accq[j] = zmc_sq_add<F>(accq[j], o[j]);
            }
        }
    }
    if (tail != 0u && ge > full_groups && lane == 0u) {
        zu32 w[4 * CG];
        const zu32 q0 = full_groups * (zu32)CG;
#pragma unroll
        for (int c = 0; c < CG; ++c) zmc_philox(q0 + (zu32)c, uc.c1, uc.c2, uc.c3, ks, &w[4 * c]);
#pragma unroll
        for (int s = 0; s < SG; ++s)
            if ((zu32)s < tail) {
                double o[NC];
                f.evalv(&w[s * D], o, nullptr);
#pragma unroll
                for (int j = 0; j < NC; ++j) acc[j] = __dadd_rn(acc[j], o[j]);
                if (SQ) {
#pragma unroll
                    for (int j = 0; j < (SQ ? NC : 1); ++j) accq[j] = zmc_sq_add<F>(accq[j], o[j]);
                }
            }
    }
#pragma unroll
    for (int j = 0; j < NC; ++j) {
        double sum = acc[j];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) sum = __dadd_rn(sum, __shfl_down_sync(0xFFFFFFFFu, sum, off));
        if (lane == 0u) a.partial[out * (zu64)NC + (zu64)j] = sum;
    }
    if (SQ) {
#pragma unroll
        for (int j = 0; j < (SQ ? NC : 1); ++j) {
            double sq = accq[j];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) sq = __dadd_rn(sq, __shfl_down_sync(0xFFFFFFFFu, sq, off));
            if (lane == 0u) a.partial_q[out * (zu64)NC + (zu64)j] = sq;
        }
    }
}

/* One (cell, trial, chunk) unit: the warp's lanes stride over the chunk's sample groups [gb, ge), lane 0 takes the ragged tail,
 * a shuffle reduction, one 8-byte store (two with SQ). */
template <class F, bool SQ>
__device__ __forceinline__ void zmc_unit(const ZmcSampleArgs& a, const F& f, const ZmcKeySchedule& ks, const ZmcUnitCounter& uc,
                                         zu32 lane, zu32 gb, zu32 ge, zu32 gfe, zu32 full_groups, zu32 tail, zu64 out) {
    constexpr int D = F::D, SG = ZmcGroup<D>::SG, CG = ZmcGroup<D>::CG;
    if constexpr (F::VEC) { zmc_unit_vec<F, SQ>(a, f, ks, uc, lane, gb, ge, gfe, full_groups, tail, out); return; }
    /* acc[0..SG) sums the groups at even multiples of 32 from the lane's first one, acc[SG..2SG) those at odd multiples --
     * whatever UNROLL is, so results do not depend on it */
    double acc[2 * SG], accq[4];     /* sums of squares: two accumulators per group in flight are enough */
#pragma unroll
    for (int s = 0; s < 2 * SG; ++s) acc[s] = 0.0;
    accq[0] = accq[1] = accq[2] = accq[3] = 0.0;
    /* EXP_QUAD with a range proof for this cell: the loop without zexp's per-sample range test; else the tested loop */
    if (F::HAS_RANGE_PROOF && f.in_range) zmc_full_groups<F, SQ, false>(f, ks, uc, gb + lane, gfe, acc, accq);
    else zmc_full_groups<F, SQ, true>(f, ks, uc, gb + lane, gfe, acc, accq);
    if (tail != 0u && ge > full_groups && lane == 0u) {   /* the partial group: only its first `tail` samples exist */
        zu32 w[4 * CG];
        const zu32 q0 = full_groups * (zu32)CG;
#pragma unroll
        for (int c = 0; c < CG; ++c) zmc_philox(q0 + (zu32)c, uc.c1, uc.c2, uc.c3, ks, &w[4 * c]);
#pragma unroll
        for (int s = 0; s < SG; ++s)
            if ((zu32)s < tail) {
                const double fv = f.eval(&w[s * D], nullptr);
                acc[s] = __dadd_rn(acc[s], fv);
                if (SQ) accq[s & 1] = zmc_sq_add<F>(accq[s & 1], fv);
            }
    }
    double sum = acc[0];
#pragma unroll
    for (int s = 1; s < 2 * SG; ++s) sum = __dadd_rn(sum, acc[s]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) sum = __dadd_rn(sum, __shfl_down_sync(0xFFFFFFFFu, sum, off));
    if (SQ) {
        double sq = __dadd_rn(__dadd_rn(accq[0], accq[1]), __dadd_rn(accq[2], accq[3]));
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) sq = __dadd_rn(sq, __shfl_down_sync(0xFFFFFFFFu, sq, off));
        if (lane == 0u) a.partial_q[out] = sq;
    }
    if (lane == 0u) a.partial[out] = sum;
}

/* UKEY: every work item has the same Philox key (n_instances == 1); it comes from the kernel
 * parameters (constant bank), so the ten round keys live in uniform registers: 20 fewer registers
 * per thread and one register operand fewer on every Philox LOP3. */
/* SQ (R13): also sum f^2 per unit, into partial_q. */
/* zmc_sample_items: the persistent item loop of one level, run by every warp of the grid until the level's counter is used up.
 * It is the body of zmc_sample_kernel and, between two grid-wide barriers, of the single-launch tree kernel (zmc_tree.cuh). */
template <class F, bool UKEY, bool SQ>
__device__ __forceinline__ void zmc_sample_items(const ZmcSampleArgs& a) {
    constexpr int D = F::D, SG = ZmcGroup<D>::SG;
    const zu32 lane = threadIdx.x & 31u;
    ZmcLevelInfo* const info = a.info;
    const zu64 n_items = info->n_items;
    const zu32 n_chunks = info->n_chunks;
    const zu32 chunk_groups = info->chunk_groups;
    const zu32 full_groups = (zu32)(a.N / (zu64)SG);       /* groups whose SG samples all exist */
    const zu32 tail = (zu32)(a.N - (zu64)full_groups * SG); /* samples in the last, partial group */
    const zu32 n_groups = full_groups + (tail ? 1u : 0u);
    const zu32 tpi = ZmcTune<F>::TRIAL_LOOP ? info->trials_per_item : 1u;

    for (;;) {
        zu64 item = 0;
        if (lane == 0) item = atomicAdd(&info->work_ctr, 1ull);
        item = __shfl_sync(0xFFFFFFFFu, item, 0);
        if (item >= n_items) break;

        ZmcUnit<D> u;
        u.template decode<ZmcTune<F>::FAST_DECODE>(a, item, n_chunks, tpi);
        F f;
        f.setup(a, u.inst, u.coords);
        ZmcKeySchedule ks;
        if (UKEY) ks.init(a.ukey[0], a.ukey[1]);
        else ks.init(a.keys[2 * u.inst], a.keys[2 * u.inst + 1]);

        /* a chunk before the last ends where the next begins ((chunk + 1) * chunk_groups <= (n_chunks - 1) * chunk_groups < n_groups);
         * the last ends with the unit. No sum that could pass 2^32, and -- measured -- the form ptxas schedules best:
         * "gb + chunk_groups < n_groups ? .. : .." in 64-bit cost 30 registers and 4 % at D = 6 */
        const zu32 gb = u.chunk * chunk_groups;
        const zu32 ge = (u.chunk + 1u < n_chunks) ? gb + chunk_groups : n_groups;
        const zu32 gfe = (ge < full_groups) ? ge : full_groups;

        if (!ZmcTune<F>::TRIAL_LOOP) {          /* the item is one unit */
            ZmcUnitCounter uc;
            uc.init(u.path_lo, u.path_hi, a.level, u.trial);
            zmc_unit<F, SQ>(a, f, ks, uc, lane, gb, ge, gfe, full_groups, tail, item);
        } else {
            /* the item's units: one, or -- trials_per_item == T -- the T trials of the cell, which share everything above */
            zu64 out = (u.cell * (zu64)a.T + u.trial) * n_chunks + u.chunk;     /* = item when trials_per_item == 1 */
            for (zu32 trial = u.trial; trial < u.trial + tpi; ++trial, ++out) {
                ZmcUnitCounter uc;
                uc.init(u.path_lo, u.path_hi, a.level, trial);
                /* opaque to the optimiser: otherwise ptxas hoists the per-cell halves of the first Philox rounds above this loop
                 * and takes 8 more registers at D = 6 */
                asm volatile("" : "+r"(uc.c1), "+r"(uc.c2), "+r"(uc.c3));
                zmc_unit<F, SQ>(a, f, ks, uc, lane, gb, ge, gfe, full_groups, tail, out);
            }
        }
    }
}

template <class F, bool UKEY, bool SQ = false>
__global__ void __launch_bounds__(ZMC_BLOCK_THREADS, ZmcTune<F>::MINB) zmc_sample_kernel(const __grid_constant__ ZmcSampleArgs a) {
    zmc_sample_items<F, UKEY, SQ>(a);
}

/* Debug kernel (parity tests P1): the first n samples of one unit through the same device functions. */
struct ZmcPointsArgs {
    ZmcSampleArgs a;        /* geometry, keys, parameters; par_* and partial unused */
    zu32 inst, trial;
    zu64 path_lo;
    zu32 path_hi;
    zu32 coords[ZMC_DEV_MAX_DIM];
    zu64 n;
    double* x;              /* [n*D] */
    double* f;              /* [n], vector-valued integrands: [n * NC], component fastest */
};

template <int D>
__device__ __forceinline__ void zmc_sample_words(zu64 s, const ZmcKeySchedule& ks, const ZmcUnitCounter& uc, zu32* w) {
    zu32 cur[4];
    zu64 have = ~0ull;
#pragma unroll
    for (int d = 0; d < D; ++d) {
        const zu64 idx = s * (zu64)D + (zu64)d;
        if ((idx >> 2) != have) { have = idx >> 2; zmc_philox((zu32)have, uc.c1, uc.c2, uc.c3, ks, cur); }
        w[d] = cur[idx & 3ull];
    }
}

/* One thread per pair of samples (2t, 2t+1). x always comes from the scalar eval(); f comes from the
 * packed eval2() for even t and from the scalar eval() for odd t, so a bit-exact comparison of f with
 * the oracle covers both code paths of the sampling kernel. */
template <class F>
__global__ void zmc_points_kernel(const __grid_constant__ ZmcPointsArgs pa) {
    constexpr int D = F::D;
    F f;
    zu32 coords[D];
#pragma unroll
    for (int d = 0; d < D; ++d) coords[d] = pa.coords[d];
    f.setup(pa.a, pa.inst, coords);
    ZmcKeySchedule ks;
    ks.init(pa.a.keys[2 * pa.inst], pa.a.keys[2 * pa.inst + 1]);
    ZmcUnitCounter uc;
    uc.init(pa.path_lo, pa.path_hi, pa.a.level, pa.trial);
    const zu64 n_pairs = (pa.n + 1ull) >> 1;
    for (zu64 t = (zu64)blockIdx.x * blockDim.x + threadIdx.x; t < n_pairs; t += (zu64)gridDim.x * blockDim.x) {
        const zu64 s0 = 2ull * t, s1 = s0 + 1ull;
        zu32 w0[D], w1[D];
        zmc_sample_words<D>(s0, ks, uc, w0);
        zmc_sample_words<D>(s1, ks, uc, w1);
        double x0[D], x1[D];
        if constexpr (F::VEC) {
            double o0[F::NC], o1[F::NC];
            f.evalv(w0, o0, x0);
            f.evalv(w1, o1, x1);
            if (pa.f) {
#pragma unroll
                for (int j = 0; j < F::NC; ++j) {
                    pa.f[s0 * F::NC + j] = o0[j];
                    if (s1 < pa.n) pa.f[s1 * F::NC + j] = o1[j];
                }
            }
        } else {
        double v0 = f.eval(w0, x0), v1 = f.eval(w1, x1);
        if ((t & 1ull) == 0ull) f.eval2(w0, w1, v0, v1);
        if (pa.f) {
            pa.f[s0] = v0;
            if (s1 < pa.n) pa.f[s1] = v1;
        }
        }
        if (pa.x) {
#pragma unroll
            for (int d = 0; d < D; ++d) {
                pa.x[s0 * D + d] = x0[d];
                if (s1 < pa.n) pa.x[s1 * D + d] = x1[d];
            }
        }
    }
}

#endif /* ZMC_DEVICE_CUH */
