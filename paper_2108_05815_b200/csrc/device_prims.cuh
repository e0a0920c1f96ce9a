// device_prims.cuh -- device primitives of the Independent algorithm.
//   2.2 primeable hash RNG       (PAPER.md 5.2.1 L693-707: prime() on (seed, location, time))
//   2.3 fixed-point -ln          (PAPER.md Eq. C.3: Exp(lambda) = -ln(U)/lambda)
//   2.4 scale by 1/(lambda*dt)
// Integer-only: every decision on the hot path is made in u32/u64 arithmetic (no libdevice, no FMA).
#pragma once
#include <stdint.h>

namespace necsim {

typedef uint32_t u32;
typedef uint64_t u64;
typedef int64_t i64;

// first twelve primes: MULT = frac(sqrt p) | 1, KEYC = frac(cbrt p), 32 bits each
#define NS_M0 0x6a09e667u
#define NS_M1 0xbb67ae85u
#define NS_M2 0x3c6ef373u
#define NS_M3 0xa54ff53bu
#define NS_M4 0x510e527fu
#define NS_M5 0x9b05688du
#define NS_M6 0x1f83d9abu
#define NS_M7 0x5be0cd19u
#define NS_M8 0xcbbb9d5du
#define NS_M9 0x629a292bu
#define NS_M10 0x9159015bu
#define NS_M11 0x152fecd9u
#define NS_C6 0x923f82a4u
#define NS_C7 0xab1c5ed5u
#define NS_C8 0xd807aa98u
#define NS_C9 0x12835b01u
#define NS_C10 0x243185beu
#define NS_C11 0x550c7dc3u
#define NS_GAMMA 0x6a09e667f3bcc909ull
#define NS_L_SPEC 0xbb67ae8584caa73bull
#define NS_L_DISP 0x3c6ef372fe94f82bull
#define NS_L_INDEX 0xa54ff53a5f1d36f1ull
#define NS_L_MIGR 0x510e527fade682d1ull
#define NS_L_COUNT 0x9b05688c2b3e6c1full
#define NS_L_THIN 0x1f83d9abfb41bd6bull
#define NS_TWO48 (1ull << 48)
#define NS_POIS_N 256u

// one Feistel round: p = a*M; (a, b) <- (hi32(p) ^ b ^ K, lo32(p))   [1 IMAD.WIDE.U32 + 1 LOP3]
__host__ __device__ __forceinline__ void feistel(u32 &a, u32 &b, u32 M, u32 K) {
    // written as separate low / high products: nvcc fuses them into ONE IMAD.WIDE.U32 (the u64 form costs an extra add)
#ifdef __CUDA_ARCH__
    const u32 lo = a * M, hi = __umulhi(a, M);
#else
    const u64 p = (u64)a * (u64)M;
    const u32 lo = (u32)p, hi = (u32)(p >> 32);
#endif
    a = hi ^ b ^ K;
    b = lo;
}

// F: fixed-key 64-bit bijection, rounds 6..11
__host__ __device__ __forceinline__ u64 hashF(u64 x) {
    u32 a = (u32)x, b = (u32)(x >> 32);
    feistel(a, b, NS_M6, NS_C6);
    feistel(a, b, NS_M7, NS_C7);
    feistel(a, b, NS_M8, NS_C8);
    feistel(a, b, NS_M9, NS_C9);
    feistel(a, b, NS_M10, NS_C10);
    feistel(a, b, NS_M11, NS_C11);
    return ((u64)a << 32) | (u64)b;
}

// two / three independent evaluations of F written round by round: the compiler emits the chains as written, and a warp
// that is alone on its scheduler then overlaps them (three in a row cost three times the latency of one)
__device__ __forceinline__ void hashF2(u64 x0, u64 x1, u64 &y0, u64 &y1) {
    u32 a0 = (u32)x0, b0 = (u32)(x0 >> 32), a1 = (u32)x1, b1 = (u32)(x1 >> 32);
    feistel(a0, b0, NS_M6, NS_C6);   feistel(a1, b1, NS_M6, NS_C6);
    feistel(a0, b0, NS_M7, NS_C7);   feistel(a1, b1, NS_M7, NS_C7);
    feistel(a0, b0, NS_M8, NS_C8);   feistel(a1, b1, NS_M8, NS_C8);
    feistel(a0, b0, NS_M9, NS_C9);   feistel(a1, b1, NS_M9, NS_C9);
    feistel(a0, b0, NS_M10, NS_C10); feistel(a1, b1, NS_M10, NS_C10);
    feistel(a0, b0, NS_M11, NS_C11); feistel(a1, b1, NS_M11, NS_C11);
    y0 = ((u64)a0 << 32) | (u64)b0; y1 = ((u64)a1 << 32) | (u64)b1;
}
__device__ __forceinline__ void hashF3(u64 x0, u64 x1, u64 x2, u64 &y0, u64 &y1, u64 &y2) {
    u32 a0 = (u32)x0, b0 = (u32)(x0 >> 32), a1 = (u32)x1, b1 = (u32)(x1 >> 32), a2 = (u32)x2, b2 = (u32)(x2 >> 32);
    feistel(a0, b0, NS_M6, NS_C6);   feistel(a1, b1, NS_M6, NS_C6);   feistel(a2, b2, NS_M6, NS_C6);
    feistel(a0, b0, NS_M7, NS_C7);   feistel(a1, b1, NS_M7, NS_C7);   feistel(a2, b2, NS_M7, NS_C7);
    feistel(a0, b0, NS_M8, NS_C8);   feistel(a1, b1, NS_M8, NS_C8);   feistel(a2, b2, NS_M8, NS_C8);
    feistel(a0, b0, NS_M9, NS_C9);   feistel(a1, b1, NS_M9, NS_C9);   feistel(a2, b2, NS_M9, NS_C9);
    feistel(a0, b0, NS_M10, NS_C10); feistel(a1, b1, NS_M10, NS_C10); feistel(a2, b2, NS_M10, NS_C10);
    feistel(a0, b0, NS_M11, NS_C11); feistel(a1, b1, NS_M11, NS_C11); feistel(a2, b2, NS_M11, NS_C11);
    y0 = ((u64)a0 << 32) | (u64)b0; y1 = ((u64)a1 << 32) | (u64)b1; y2 = ((u64)a2 << 32) | (u64)b2;
}

struct SeedKey {
    u32 K[6];
};

// host side key schedule: h = F(seed); K[r] = hi32(F(h + (r+1)*GAMMA))
static inline SeedKey key_schedule(u64 seed) {
    SeedKey sk;
    u64 h = hashF(seed);
    for (int r = 0; r < 6; ++r) sk.K[r] = (u32)(hashF(h + (u64)(r + 1) * NS_GAMMA) >> 32);
    return sk;
}

// prime(loc, k): keyed rounds 0..5 on (a, b) = (loc, k)
__device__ __forceinline__ u64 prime(const SeedKey &sk, u32 loc, u32 k) {
    u32 a = loc, b = k;
    feistel(a, b, NS_M0, sk.K[0]);
    feistel(a, b, NS_M1, sk.K[1]);
    feistel(a, b, NS_M2, sk.K[2]);
    feistel(a, b, NS_M3, sk.K[3]);
    feistel(a, b, NS_M4, sk.K[4]);
    feistel(a, b, NS_M5, sk.K[5]);
    return ((u64)a << 32) | (u64)b;
}

// draws for the event candidate at stream position X = s + j*GAMMA
__device__ __forceinline__ u64 draw_time(u64 X) { return hashF(X); }
__device__ __forceinline__ u64 draw_spec(u64 X) { return hashF(X ^ NS_L_SPEC); }
__device__ __forceinline__ u64 draw_disp(u64 X, u32 r) { return hashF((X ^ NS_L_DISP) + (u64)r * NS_GAMMA); }
__device__ __forceinline__ u64 draw_index(u64 X) { return hashF(X ^ NS_L_INDEX); }
__device__ __forceinline__ u64 draw_migr(u64 X) { return hashF(X ^ NS_L_MIGR); }

__device__ __forceinline__ u64 mulhi64(u64 x, u64 n) { return __umul64hi(x, n); }
// (x * d) >> 64 for a 32-bit d: two 32x32 products instead of a full 64x64
__device__ __forceinline__ u32 mulhi64_u32(u64 x, u32 d) {
    u64 lo = (u64)(u32)x * (u64)d;
    u64 hi = (u64)(u32)(x >> 32) * (u64)d + (lo >> 32);
    return (u32)(hi >> 32);
}
__device__ __forceinline__ bool bern(u64 x, u64 thr) { return (x >> 11) < thr; }

// Shared-memory reads by 32-bit shared-window address. Tables handed to device functions as generic pointers make the
// compiler rebuild the window base (S2R + LEA) at every access; a plain address register does not.
struct SmemTables {
    u32 q, a;      // -ln tables: Q[512] u16, A[512] u64
    u32 tg, g2;    // rounded-normal thresholds u32[<=1024], guide uint2[2048]
    u32 pc, pg;    // Poisson cdf thresholds u64[256], guide u16[256] on the top byte of the draw
};
__device__ __forceinline__ u32 smem_addr(const void *p) {
    u32 a = (u32)__cvta_generic_to_shared(p), r;
    asm volatile("mov.u32 %0, %1;" : "=r"(r) : "r"(a));   // opaque: keep the address in a register, do not rebuild it per access
    return r;
}
__device__ __forceinline__ u32 lds_u16(u32 addr) { u32 v; asm("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(addr)); return v; }
__device__ __forceinline__ u32 lds_u32(u32 addr) { u32 v; asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr)); return v; }
__device__ __forceinline__ u64 lds_u64(u32 addr) { u64 v; asm("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(addr)); return v; }
__device__ __forceinline__ uint2 lds_v2(u32 addr) { uint2 v; asm("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr)); return v; }

// fixed-point -ln: Q8.56 of -ln(U), U = M * 2^-(z+50). Tables: 512 entries in shared memory
#define NS_LN2_56 49946518145322873ull
__device__ __forceinline__ u64 neglog(u64 x, const SmemTables &sm) {
    u32 z = (u32)__clzll((long long)x);         // 64 for x = 0
    u64 y = (z >= 64) ? 0ull : (x << z);
    u64 M = (y >> 14) | 1ull;
    u32 i = (u32)(y >> 54) & 511u;
    u64 P = M * (u64)lds_u16(sm.q + 2u * i);
    u64 r = P & ((1ull << 61) - 1);
    u32 t = (u32)(r >> 21);
    u32 h1 = 0x55555555u - (t >> 10);
    u32 h2 = 0x80000000u - (__umulhi(t, h1) >> 8);
    u64 u = (u64)__umulhi(t, h2);
    u64 c = ((u64)t * u) >> 24;
    u64 G = lds_u64(sm.a + 8u * i) + ((r >> 5) - c);
    u64 Lz = (u64)(z + 1) * NS_LN2_56;
    return Lz > G ? Lz - G : 0ull;
}

// Poisson sampler: N = #{n : c >= PC[n]}, c = F(s ^ L_COUNT). pg[b] = #{n : PC[n] < b << 56} starts a short
// forward scan over the non-decreasing thresholds.
__device__ __forceinline__ u32 poisson_count_of(u64 c, const SmemTables &sm) {   // c = F(s ^ L_COUNT)
    u32 n = lds_u16(sm.pg + 2u * (u32)(c >> 56));
    while (n < NS_POIS_N && lds_u64(sm.pc + 8u * n) <= c) ++n;
    return n;
}
__device__ __forceinline__ u32 poisson_count(u64 s, const SmemTables &sm) {
    const u64 c = hashF(s ^ NS_L_COUNT);
    u32 n = lds_u16(sm.pg + 2u * (u32)(c >> 56));
    while (n < NS_POIS_N && lds_u64(sm.pc + 8u * n) <= c) ++n;
    return n;
}
// offset of point X and whether it exists for a cell with thinning threshold `thin`
__device__ __forceinline__ u64 poisson_offset(u64 X) { return hashF(X) >> 16; }
__device__ __forceinline__ bool poisson_kept(u64 X, u32 thin) { return thin == 0xFFFFFFFFu || (u32)hashF(X ^ NS_L_THIN) < thin; }

// E / mu in Q16.48: bits of the exact 96-bit product E * Cm
__device__ __forceinline__ u64 scale_exp(u64 E, u32 Cm, u32 sh) {
    u64 Eh = E >> 32, El = E & 0xFFFFFFFFull;
    return ((Eh * (u64)Cm) + ((El * (u64)Cm) >> 32)) >> sh;
}

// real time of (k, f): ((double)k + (double)f * 2^-48) * delta_t, no contraction
__device__ __forceinline__ double event_time(u32 k, u64 f, double delta_t) {
    double a = __dmul_rn((double)f, 0x1p-48);
    double b = __dadd_rn((double)k, a);
    return __dmul_rn(b, delta_t);
}

// 128-bit atomic exchange in global memory (PTX ISA 8.3+, sm_90+): returns the previous 16 bytes
__device__ __forceinline__ uint4 atomic_exch_128(uint4 *addr, uint4 v) {
    u64 lo = ((u64)v.y << 32) | v.x, hi = ((u64)v.w << 32) | v.z, olo, ohi;
    asm volatile(
        "{\n\t"
        ".reg .b128 vin, vout;\n\t"
        "mov.b128 vin, {%2, %3};\n\t"
        "atom.global.relaxed.gpu.exch.b128 vout, [%4], vin;\n\t"
        "mov.b128 {%0, %1}, vout;\n\t"
        "}"
        : "=l"(olo), "=l"(ohi)
        : "l"(lo), "l"(hi), "l"(addr)
        : "memory");
    return make_uint4((u32)olo, (u32)(olo >> 32), (u32)ohi, (u32)(ohi >> 32));
}

// the same exchange under a predicate, the result landing in (olo, ohi) only where it executes: no branch around it and no
// copy of the result after it, so that a caller which consumes the result much later does not wait for the round trip here
__device__ __forceinline__ void atomic_exch_128_if(bool p, uint4 *addr, uint4 v, u64 &olo, u64 &ohi) {
    const u64 lo = ((u64)v.y << 32) | v.x, hi = ((u64)v.w << 32) | v.z;
    asm volatile(
        "{\n\t"
        ".reg .pred q;\n\t"
        ".reg .b128 vin, vout;\n\t"
        "setp.ne.u32 q, %4, 0;\n\t"
        "mov.b128 vin, {%2, %3};\n\t"
        "mov.b128 vout, {%0, %1};\n\t"
        "@q atom.global.relaxed.gpu.exch.b128 vout, [%5], vin;\n\t"
        "mov.b128 {%0, %1}, vout;\n\t"
        "}"
        : "+l"(olo), "+l"(ohi)
        : "l"(lo), "l"(hi), "r"((u32)p), "l"(addr)
        : "memory");
}

}  // namespace necsim
