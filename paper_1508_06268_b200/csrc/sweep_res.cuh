// sweep_res.cuh -- the shared-memory-resident sweep: every lattice plane stays in the shared memory of
// one SM for a whole launch (all phases of an exchange period).  DESIGN.md section 6.
//
// Decomposition.  The D*n active replicas (by temperature rank) are stacked into one list of
// D*n*L planes (plane P = (d*n + t)*L + z; a replica shard lists its stored slots instead of the ranks).  CTA b of a cooperative launch owns the contiguous run
// [start_b, start_b + count_b) with counts differing by at most one (the last CTAs take the longer runs), so 148 SMs hold 55 or 56 planes
// each at L = 64, R = 128: no replica-granular imbalance (128 replicas do not divide over 148 SMs).
// A run is loaded once, swept 2*sweeps phases (colour 0, colour 1, ...) in place, and stored once.
// Only the planes at the ends of a run (and at a replica seam inside it) have a z-neighbour in
// another CTA: after every phase their freshly written colour is also stored to global memory and
// the CTA's progress word is released; the neighbour acquires it before it reads those rows
// straight from L2.  Boundary planes are processed first in every phase, so the neighbour has a
// whole phase of slack.  All CTAs are co-resident (cooperative launch), hence no deadlock.
//
// Inside a CTA there is no barrier between phases either.  Work is cut into warp tasks (phase, 32-row
// block: both checkerboard classes of those rows); warps draw task numbers from one shared counter
// (phase-major), and a task starts as soon as the blocks holding its own plane and its two z-neighbour
// planes have finished the previous phase (per-block completion counters in shared memory).  A task
// only ever waits for lower-numbered tasks, so the lowest outstanding task can always run: no
// deadlock, no tail at the end of a phase.
//
// Measurement (S5) rides on the last phase of the launch (colour 1), from registers the update
// holds anyway: Msum and Ef of the colour-1 words it has just updated and of the colour-0 words of the same
// row (final since the phase before; only their field is loaded in addition), and since every bond has
// exactly one colour-1 end, Eb = sum over colour-1 sites of s_i' * (six-neighbour sum).  Sums go per replica to shared memory,
// then to View::acc with integer atomics (order-independent, hence deterministic).  The
// CTA that finishes last then runs the exchange step itself (small batches), so a whole
// parallel-tempering move is one launch.
//
// Several moves per launch (the MULTI instantiation; single realisation, not sharded).  A call that spans several exchange periods
// keeps the run in shared memory across them: at the end of a period the CTAs hand their sums over, meet at an arrival counter,
// the last one to arrive runs the exchange step and releases a flag word, and every CTA re-reads the ranks of its resident slots
// (lattices never move: only the per-replica tables change) before the task flow goes on with the next period's phases.
//
// In shared memory a spin is a byte holding 0 or SP (= 8), four same-colour sites per 32-bit word
// exactly as in global memory (where it is 0/1), so the six-neighbour count of four sites is a few
// IADD3, and count*SP + spin*8*SP [+ field bit] is directly the byte offset of the site's entry in
// the replica's 8-byte acceptance table: one PRMT splices it into the (256-byte aligned) table
// address, one LDS.64 fetches the entry.
//
// A thread owns one row of one colour (L/2 sites = 4K words = 4K Philox calls) and walks it one
// 16-site piece at a time; the 32 lanes of a warp own 32 rows of the same checkerboard class
// s = (y+z)&1, so the direction of the second x-neighbour ((s+colour)&1) is warp-uniform.  Shared
// memory is laid out [colour][s][piece][row] with a compile-time row capacity, which makes every
// 16-byte access of a warp contiguous (no bank conflicts) and every array offset an immediate; the
// field is read from a copy stored in the same task order (coalesced 16-byte loads from L2).
#pragma once
#include <cstdint>
#include "kernels_ref.cuh"
#include "philox.cuh"
#include "sweep_flow.cuh"
#include "view.h"

namespace rfim {

// RFIM_RES_TIMING (debug builds): globaltimer stamps of the kernel's stages per CTA -- 0 start, 1 set-up done, 2 run loaded,
// 3 task loop done (warp 0), 4 after the barrier, 5 run stored, 6 end -- read back with rfim_pt_debug_timing
// (bench.py --stage-timing; profiles/r2_res_stage_timing.md)
#ifdef RFIM_RES_TIMING
__device__ unsigned long long g_res_timing[256][8];
__device__ __forceinline__ unsigned long long res_now() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#define RES_STAMP(i) do { if (threadIdx.x == 0) g_res_timing[blockIdx.x][i] = res_now(); } while (0)
#else
#define RES_STAMP(i) do { } while (0)
#endif

// RFIM_RES_CHECK (debug builds; compute-sanitizer is not available on the GPU pool): every shared-memory row address, global
// spin offset, field index and progress value the kernel forms is range-checked; a violation sets bit 1 of diag[0], which
// every synchronising getter reports as an error (profiles/r2_sanitizer.md).
#ifdef RFIM_RES_CHECK
#define RES_CHECK(cond) do { if (!(cond)) atomicOr(rp.diag, 2ull); } while (0)
#else
#define RES_CHECK(cond) do { } while (0)
#endif

#ifndef RFIM_RES_THREADS
#define RFIM_RES_THREADS 512
#endif
constexpr int kResThreads = RFIM_RES_THREADS;
constexpr uint32_t kResSP = 8;                  // shared-memory spin coding: 0 / SP
constexpr int kResTabBytes = 256;               // per-replica acceptance table slot (256-byte aligned)
constexpr int kResLoadDepth = 8;                // 16-byte loads a thread keeps in flight while the run is loaded

// shared-memory geometry of the resident kernel for L = 32 K
template <int K>
struct ResGeom {
    static constexpr int L = 32 * K;
    static constexpr int LH = L / 2;                        // rows per class per plane
    static constexpr int ROWB = 16 * K;                     // bytes (= sites) per row per colour
    static constexpr int W = 4 * K;                         // words (= Philox calls) per row
    static constexpr int MAXPLANES = K == 2 ? 56 : 221;     // planes one CTA can hold (227 KB of shared memory)
    static constexpr int ECAP = MAXPLANES * LH;             // rows per (colour, class, piece) array
    static constexpr int ARR = ECAP * 16;                   // bytes per array
    static constexpr int SPINS_BYTES = 4 * K * ARR;         // [colour][class][piece][row] uint4
    static constexpr int NBCAP = (ECAP + 31) / 32;          // 32-row blocks
};
__host__ __device__ constexpr int res_max_planes(int L) { return L == 64 ? ResGeom<2>::MAXPLANES : ResGeom<1>::MAXPLANES; }

struct ResParams {
    int phases;                  // 2 * sweeps of this launch, <= 254
    int measure;                 // != 0: the last phase also measures (Eb, Ef, Msum -> View::acc)
    int exchange;                // != 0: the CTA that finishes last runs the exchange step of every member
    int nact;                    // CTAs that own planes
    uint32_t xstep;              // exchange step index, time-series row, record flag (exchange != 0)
    long long xrow;
    uint32_t* ticket;            // arrival counter of the fused exchange (left at zero)
    uint32_t sweep0;             // global sweep index of phase 0
    uint32_t epoch;              // launch id: progress words hold (epoch << 8) | phases published
    uint32_t* prog;              // [grid]
    int total_planes;            // D * n * L
    int q, rem;                  // run of CTA b: count = q, or q + 1 for the last rem CTAs of the grid
    int cap_reps;                // replicas a run can touch -- same carve for every CTA
    int d0;                      // first member of this launch's group (plane P = ((d - d0) * n + t) * L + z)
    const float* fielda_res;     // Gaussian: [D][2][L][2][4K][L/2] float4 (task order), (float)g_i (exact)
    const uint8_t* fieldb_res;   // bimodal:  [D][2][L][2][K][L/2] uint4, 0x80 where h_i = +1
    const long long* gsum;       // Gaussian: [D][L] sum of g_i over plane z
    unsigned long long* diag;
    // several parallel-tempering moves per launch (MULTI instantiation only): the launch ends on an exchange step and holds
    // nseg of them, after phase first2 - 1, first2 + period2 - 1, ...; the run stays in shared memory across them
    int nseg, first2, period2;
    uint32_t* xflag;             // release word of the mid-launch exchange steps: (epoch << 8) | steps done
    uint32_t rk0[20];            // Philox round keys of member 0 (used from the constant bank when D == 1)
};

struct ResPlane {                // 8 bytes per resident plane
    int16_t zp_pl, zm_pl;        // local index of plane z+1 / z-1, or -1: it lives in another CTA
    uint8_t zp_owner, zm_owner;  // that CTA
    uint8_t rep, z;
};

struct ResRep {                  // per replica touched by the run
    int ds, d, slot, tr;
    float band; uint32_t never;
    double beta;
    uint32_t rk[20];             // Philox round keys rk[2r] = k0 + r*W0, rk[2r+1] = k1 + r*W1
};

__host__ __device__ inline size_t res_smem_bytes(int L, int cap_reps) {
    const size_t spins = L == 64 ? ResGeom<2>::SPINS_BYTES : ResGeom<1>::SPINS_BYTES;
    const size_t maxpl = L == 64 ? ResGeom<2>::MAXPLANES : ResGeom<1>::MAXPLANES;
    const size_t nbcap = L == 64 ? ResGeom<2>::NBCAP : ResGeom<1>::NBCAP;
    size_t b = spins + (size_t)cap_reps * kResTabBytes;
    b += (size_t)cap_reps * sizeof(ResRep);
    b += maxpl * sizeof(ResPlane);
    b += nbcap * 2 * sizeof(int);                           // block order, block completion counters
    b += 16;                                                // counters
    b += (size_t)cap_reps * 3 * sizeof(long long);          // measurement accumulators
    b += (size_t)(kResThreads / 32) * 4 * sizeof(long long); // per-warp measurement slots
    return (b + 15) & ~(size_t)15;
}

__device__ __forceinline__ uint32_t lds32(uint32_t saddr) {
    uint32_t r;
#if defined(__CUDA_ARCH__)
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(saddr));
#else
    r = 0;
#endif
    return r;
}

__device__ __forceinline__ uint2 lds64(uint32_t saddr) {
    uint2 r;
#if defined(__CUDA_ARCH__)
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(saddr));
#else
    r.x = r.y = 0;
#endif
    return r;
}

// prmt.b32 in its default mode: selector nibble n picks byte (n & 7) of {b, a}; bit 3 replicates that byte's sign
// bit over the whole byte (the CUDA intrinsic __byte_perm ignores bit 3)
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t r;
#if defined(__CUDA_ARCH__)
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
#else
    r = 0;
#endif
    return r;
}

__device__ __forceinline__ int lds_volatile(const int* p) { return *reinterpret_cast<const volatile int*>(p); }

// per-block completion counters (shared memory, CTA scope): a task's rows are stored before its counter is bumped with
// release semantics, and a reader that has seen the count with an acquire load may read those rows -- no separate fence
// on the reading side (the acquire load compiles to a plain LDS; shared-memory accesses of a warp are issued in order)
__device__ __forceinline__ int lds_acquire(const int* p) {
    int v;
#if defined(__CUDA_ARCH__)
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(p)) : "memory");
#else
    v = *p;
#endif
    return v;
}
__device__ __forceinline__ void sts_release_inc(int* p) {
#if defined(__CUDA_ARCH__)
    asm volatile("red.release.cta.shared.add.u32 [%0], 1;" :: "r"((uint32_t)__cvta_generic_to_shared(p)) : "memory");
#else
    ++*p;
#endif
}

// ---- one 16-site piece between its global form (16 bytes of 0/1, or 16 bits when View::packed) and the shared-memory
// form (16 bytes of 0/SP).  `off` is the piece's index in spins (a multiple of 16).
__device__ __forceinline__ uint32_t res_nibble_to_word(uint32_t nib) { return ((nib & 0xFu) * 0x00204081u) & 0x01010101u; }
__device__ __forceinline__ uint32_t res_word_to_nibble(uint32_t w01) { return (((w01 & 0x01010101u) * 0x01020408u) >> 24) & 0xFu; }
__device__ __forceinline__ uint4 res_piece_from_global(const uint8_t* spins, size_t off, int packed) {
    uint4 x;
    if (packed) {
#if defined(__CUDA_ARCH__)
        const uint32_t q = __ldcg(reinterpret_cast<const unsigned short*>(spins + (off >> 3)));
#else
        const uint32_t q = 0;
#endif
        x.x = res_nibble_to_word(q); x.y = res_nibble_to_word(q >> 4); x.z = res_nibble_to_word(q >> 8); x.w = res_nibble_to_word(q >> 12);
    } else {
        x = ld_cg16(spins + off);
    }
    x.x *= kResSP; x.y *= kResSP; x.z *= kResSP; x.w *= kResSP;
    return x;
}
// raw form of a piece as it sits in global memory (16 bytes, or 16 bits in .x when packed) and its conversion
__device__ __forceinline__ uint4 res_piece_raw(const uint8_t* spins, size_t off, int packed) {
    uint4 x = make_uint4(0u, 0u, 0u, 0u);
    if (packed) {
#if defined(__CUDA_ARCH__)
        x.x = __ldcg(reinterpret_cast<const unsigned short*>(spins + (off >> 3)));
#endif
    } else {
        x = ld_cg16(spins + off);
    }
    return x;
}
__device__ __forceinline__ uint4 res_piece_expand(uint4 x, int packed) {
    if (packed) {
        const uint32_t q = x.x;
        x.x = res_nibble_to_word(q); x.y = res_nibble_to_word(q >> 4); x.z = res_nibble_to_word(q >> 8); x.w = res_nibble_to_word(q >> 12);
    }
    x.x *= kResSP; x.y *= kResSP; x.z *= kResSP; x.w *= kResSP;
    return x;
}
__device__ __forceinline__ void res_piece_to_global(uint8_t* spins, size_t off, int packed, uint4 x) {
    x.x >>= 3; x.y >>= 3; x.z >>= 3; x.w >>= 3;
    if (packed)
        *reinterpret_cast<unsigned short*>(spins + (off >> 3)) = (unsigned short)(res_word_to_nibble(x.x) | (res_word_to_nibble(x.y) << 4) |
                                                                                  (res_word_to_nibble(x.z) << 8) | (res_word_to_nibble(x.w) << 12));
    else
        *reinterpret_cast<uint4*>(spins + off) = x;
}

__device__ __forceinline__ Words4 philox_rkreg(const uint32_t (&rk)[20], uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(kPhiloxM0, c0), lo0 = kPhiloxM0 * c0;
        const uint32_t hi1 = __umulhi(kPhiloxM1, c2), lo1 = kPhiloxM1 * c2;
        const uint32_t n0 = hi1 ^ c1 ^ rk[2 * r];
        const uint32_t n2 = hi0 ^ c3 ^ rk[2 * r + 1];
        c1 = lo1; c3 = lo0; c0 = n0; c2 = n2;
    }
    Words4 w;
    w.w0 = c0; w.w1 = c1; w.w2 = c2; w.w3 = c3;
    return w;
}

// u as a float, rounded toward minus infinity: cvt.rm compiles to I2F.U32.RM, which runs on the XU pipe (the default
// round-to-nearest conversion is I2FP on the ALU pipe, the pipe the Philox XORs already saturate).  Error < 2^-23 relative.
__device__ __forceinline__ float res_u2f(uint32_t u) {
#if defined(__CUDA_ARCH__)
    float f;
    asm("cvt.rm.f32.u32 %0, %1;" : "=f"(f) : "r"(u));
    return f;
#else
    return (float)u;
#endif
}

// the float path of one Gaussian attempt: d = float(u) - P~, P~ = 2^(g*y + x); accept iff d < 0 unless |d| < band
__device__ __forceinline__ float res_gauss_diff(uint32_t idx8, int j, uint32_t tab_addr, float a, uint32_t u) {
    const uint2 ent = lds64(__byte_perm(idx8, tab_addr, 0x7650 + j));
    const float P = ex2_approx(fmaf(a, __uint_as_float(ent.y), __uint_as_float(ent.x)));
    return res_u2f(u) - P;
}

// Rare path: some site of the piece fell inside the float path's guard band.  Redo the piece's four words: sites
// outside the band keep the float decision (the same operations, hence the same bits), sites inside it take the
// exact binary64 rule of DESIGN.md S3.  idx8 = table-offset bytes before the update (SP*n1 + 8*SP*s).
__device__ __noinline__ uint4 res_gauss_piece_fix(const View& v, uint4 idx8v, uint32_t tab_addr, float band, const float4* __restrict__ fa,
                                                  int fa_stride, const int32_t* __restrict__ g16, const ResRep* rr, uint32_t q,
                                                  uint32_t sweep, uint32_t dom) {
    const uint32_t idx8[4] = {idx8v.x, idx8v.y, idx8v.z, idx8v.w};
    uint32_t out[4];
    for (int w = 0; w < 4; ++w) {
        const Words4 r = philox4x32_10(rr->rk[0], rr->rk[1], q + (uint32_t)w, sweep, (uint32_t)rr->slot, dom);
        const uint32_t u[4] = {r.w0, r.w1, r.w2, r.w3};
        const float4 f4 = __ldg(fa + (long long)w * fa_stride);
        const float a[4] = {f4.x, f4.y, f4.z, f4.w};
        uint32_t me = (idx8[w] >> 3) & (kResSP * 0x01010101u);
        for (int j = 0; j < 4; ++j) {
            const float d = res_gauss_diff(idx8[w], j, tab_addr, a[j], u[j]);
            bool acc = d < 0.0f;
            if (fabsf(d) < band) {
                const uint32_t bb = (idx8[w] >> (8 * j)) & 0xFFu;
                acc = gauss_accept_exact(v, (int)(bb >> 6), (int)((bb >> 3) & 7u), g16[4 * w + j], rr->beta, u[j]);
            }
            if (acc) me ^= kResSP << (8 * j);
        }
        out[w] = me;
    }
    return make_uint4(out[0], out[1], out[2], out[3]);
}

// slow side of a task's dependency wait (the fast check failed, or a neighbour plane lives in another CTA)
__device__ __noinline__ void res_wait_slow(const int* s_done, int eb, int b_zp, int b_zm, int p, const uint32_t* prog_p,
                                           const uint32_t* prog_m, uint32_t want, unsigned long long* diag) {
    int spins = 0;
    for (;;) {
        bool ok = lds_acquire(s_done + eb) >= p && lds_acquire(s_done + b_zp) >= p && lds_acquire(s_done + b_zm) >= p;
        if (prog_p) ok = ok && (int32_t)(ld_acquire_gpu(prog_p) - want) >= 0;
        if (prog_m) ok = ok && (int32_t)(ld_acquire_gpu(prog_m) - want) >= 0;
        if (__all_sync(0xFFFFFFFFu, ok)) break;
        backoff();
        if (++spins > (1 << 22)) { if ((threadIdx.x & 31) == 0) atomicOr(diag, 1ull); break; }
    }
}

// one 16-site piece of a row: own word, same-row words of the other colour, and ns = SP * (number of up neighbours)
struct ResPiece { uint32_t me[4], cw[4], ns[4]; };

// rem: where the rows of a z-neighbour plane that lives in another CTA are found in global memory (boundary tasks only)
struct ResRemote { const uint8_t* spins; size_t off_p, off_m; bool any, p, m; int packed; };   // 64-bit: the spin buffer can exceed 2^32 sites

// xr: the row's words of the other colour (all K pieces, loaded once per row: the far x-neighbour of a piece's edge
// byte is a word of the neighbouring piece, periodic in x)
template <int K>
__device__ __forceinline__ ResPiece res_load_piece(const uint8_t* smem, const uint4 (&xr)[K], uint32_t a_yp, uint32_t a_ym, uint32_t a_zp,
                                                   uint32_t a_zm, uint32_t a_me, int k, int dir, const ResRemote& rem) {
    constexpr int ARR = ResGeom<K>::ARR;
    const uint4 x = xr[k];
    const uint4 yp = *reinterpret_cast<const uint4*>(smem + a_yp + k * ARR);
    const uint4 ym = *reinterpret_cast<const uint4*>(smem + a_ym + k * ARR);
    uint4 zp = *reinterpret_cast<const uint4*>(smem + a_zp + k * ARR);
    uint4 zm = *reinterpret_cast<const uint4*>(smem + a_zm + k * ARR);
    const uint4 m = *reinterpret_cast<const uint4*>(smem + a_me + k * ARR);
    if (rem.any) {                                  // warp-uniform: only boundary tasks come here
        if (rem.p) zp = res_piece_from_global(rem.spins, rem.off_p + 16u * k, rem.packed);
        if (rem.m) zm = res_piece_from_global(rem.spins, rem.off_m + 16u * k, rem.packed);
    }
    const uint32_t edge = dir == 0 ? xr[(k + K - 1) % K].w : xr[(k + 1) % K].x;
    ResPiece pc;
    pc.me[0] = m.x; pc.me[1] = m.y; pc.me[2] = m.z; pc.me[3] = m.w;
    pc.cw[0] = x.x; pc.cw[1] = x.y; pc.cw[2] = x.z; pc.cw[3] = x.w;
    pc.ns[0] = yp.x + ym.x + zp.x + zm.x + x.x; pc.ns[1] = yp.y + ym.y + zp.y + zm.y + x.y;
    pc.ns[2] = yp.z + ym.z + zp.z + zm.z + x.z; pc.ns[3] = yp.w + ym.w + zp.w + zm.w + x.w;
    if (dir == 0) {
        pc.ns[0] += __funnelshift_r(edge, pc.cw[0], 24);
#pragma unroll
        for (int w = 1; w < 4; ++w) pc.ns[w] += __funnelshift_r(pc.cw[w - 1], pc.cw[w], 24);
    } else {
#pragma unroll
        for (int w = 0; w < 3; ++w) pc.ns[w] += __funnelshift_r(pc.cw[w], pc.cw[w + 1], 8);
        pc.ns[3] += __funnelshift_r(pc.cw[3], edge, 8);
    }
    return pc;
}

// Measurement partials of one 16-site piece in the last phase of a launch (out of line: the measuring instantiation must not
// add to the register pressure of the row update).  me = the colour-1 words just updated, idx8 = their table offsets before
// the update (bits 3..5 of a byte = SP * n1), c0 = the colour-0 words of the same row and piece; f1 / f0 = the field of the
// two (bimodal: one uint4 of 0x80 flags; Gaussian: four float4 `stride` apart, g_i exact).  Returns {64 sum s n1 over the
// colour-1 sites, packed byte sums of the eight words (SP per up spin), field term, bimodal: number of h_i = +1 sites}:
// field term = SP sum hb s (bimodal) or the sum of g_i over the up spins (Gaussian, |.| <= 32 * 2^23), both colours.
template <int KIND>
__device__ __noinline__ int4 res_measure_piece(uint4 mev, uint4 idx8v, uint4 c0v, const void* f1, const void* f0, int stride) {
    const uint32_t me[4] = {mev.x, mev.y, mev.z, mev.w}, c0[4] = {c0v.x, c0v.y, c0v.z, c0v.w};
    const uint32_t ix[4] = {idx8v.x, idx8v.y, idx8v.z, idx8v.w};
    int sn = 0, ef = 0, hh = 0;
    uint32_t ws = 0;
    if (KIND == 0) {
        const uint4 b1 = __ldg(static_cast<const uint4*>(f1)), b0 = __ldg(static_cast<const uint4*>(f0));
        const uint32_t h1[4] = {b1.x >> 7, b1.y >> 7, b1.z >> 7, b1.w >> 7}, h0[4] = {b0.x >> 7, b0.y >> 7, b0.z >> 7, b0.w >> 7};   // 0/1 per byte
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            sn += dot4(me[w], ix[w] & 0x38383838u);
            ws += me[w] + c0[w];
            ef += dot4(h1[w], me[w]) + dot4(h0[w], c0[w]);
            hh += dot4(h1[w] + h0[w], 0x01010101u);
        }
    } else {
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const float4 a1 = __ldg(static_cast<const float4*>(f1) + (long long)w * stride), a0 = __ldg(static_cast<const float4*>(f0) + (long long)w * stride);
            const float g1[4] = {a1.x, a1.y, a1.z, a1.w}, g0[4] = {a0.x, a0.y, a0.z, a0.w};
            sn += dot4(me[w], ix[w] & 0x38383838u);
            ws += me[w] + c0[w];
            const uint32_t s1 = me[w] >> 3, s0 = c0[w] >> 3;                               // 0/1 per byte
#pragma unroll
            for (int j = 0; j < 4; ++j)
                ef += __float2int_rn(g1[j]) * (int)__byte_perm(s1, 0u, 0x4440 + j) + __float2int_rn(g0[j]) * (int)__byte_perm(s0, 0u, 0x4440 + j);
        }
    }
    return make_int4(sn, (int)ws, ef, hh);
}

__device__ __noinline__ void res_flush_sums(long long* s_acc, int rep, long long eb, long long ef, long long ms) {
    if (rep < 0) return;
    atomicAdd(reinterpret_cast<unsigned long long*>(s_acc + 3 * rep + 0), (unsigned long long)eb);
    atomicAdd(reinterpret_cast<unsigned long long*>(s_acc + 3 * rep + 1), (unsigned long long)ef);
    atomicAdd(reinterpret_cast<unsigned long long*>(s_acc + 3 * rep + 2), (unsigned long long)ms);
}

// Per-task lane constants of the row update: shared-memory byte offsets of class 0 (class 1 = + K * ARR, an
// immediate), everything else the two rows of a task share.
struct ResLane {
    uint32_t me, x;              // my row in my colour / in the other colour, class 0
    uint32_t ya, yb, yc;         // rows i+1, i, i-1 of my plane in the other colour, class 0 (periodic in y)
    uint32_t zp, zm;             // row i of the z-neighbour planes in the other colour, class 0
    uint32_t q00;                // Philox counter word of (y = 2i, xh = 0)
    uint32_t slot, tab_addr;
    float band;
    uint32_t zpar;               // z & 1
    const float4* fp0;           // Gaussian field of (colour, plane, class 0), row i
    const uint4* fq0;            // bimodal field, same place
    uint32_t grow0;              // BND / rare path: byte offset of row y = 2i of colour c inside the slot's lattice
    uint32_t ds2, d2;
};

// One row (L/2 same-colour sites) of one checkerboard class S: K pieces of 16 sites.  DIR (warp-uniform): the
// second x-neighbour sits at xh-1 (0) or xh+1 (1).  BND: a z-neighbour plane lives in another CTA (rows read from and
// published to global memory); MEAS: also measure; RAGGED: lanes past the last row redo it and do not store.
template <int KIND, int K, bool NEVER, bool UNI, bool BND, bool MEAS, bool RAGGED, bool FLATE = true>
__device__ __forceinline__ void res_row(const View& v, const ResParams& rp, uint8_t* smem, const ResLane& ln, const int s, const int c, const int DIR,
                                        const uint32_t sweep, const uint32_t dom, const ResRep* rr, const bool valid,
                                        const bool remote_p, const bool remote_m, const size_t roff_p, const size_t roff_m,
                                        long long& m_eb, long long& m_ef, long long& m_ms) {
    using G = ResGeom<K>;
    constexpr int LH = G::LH, ROWB = G::ROWB, W = G::W, ARR = G::ARR;
    const uint32_t ys = (uint32_t)s ^ ln.zpar;
    const uint32_t sK = s ? (uint32_t)(K * ARR) : 0u, tK = (uint32_t)(K * ARR) - sK;
    const uint32_t a_me = ln.me + sK, a_x = ln.x + sK;
    const uint32_t a_yp = (ys ? ln.ya : ln.yb) + tK, a_ym = (ys ? ln.yb : ln.yc) + tK;
    const uint32_t a_zp = ln.zp + tK, a_zm = ln.zm + tK;
    const uint32_t q0 = ln.q00 + (ys ? W : 0);
    const float4* fp = ln.fp0 + (s ? W * LH : 0);
    const uint4* fq = ln.fq0 + (s ? K * LH : 0);
    const uint32_t grow = ln.grow0 + (ys ? ROWB : 0);          // only BND and the rare exact path use it
    ResRemote rem;
    rem.spins = v.spins; rem.any = BND; rem.p = BND && remote_p; rem.m = BND && remote_m; rem.packed = v.packed;
    rem.off_p = roff_p + (ys ? ROWB : 0); rem.off_m = roff_m + (ys ? ROWB : 0);

    uint32_t rk[20];
    if (UNI) {
#pragma unroll
        for (int j = 0; j < 20; ++j) rk[j] = rp.rk0[j];
    } else {
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            const uint4 q4 = reinterpret_cast<const uint4*>(rr->rk)[j];
            rk[4 * j] = q4.x; rk[4 * j + 1] = q4.y; rk[4 * j + 2] = q4.z; rk[4 * j + 3] = q4.w;
        }
    }

    RES_CHECK(a_me + (K - 1) * ARR + 16 <= (uint32_t)G::SPINS_BYTES && a_x + (K - 1) * ARR + 16 <= (uint32_t)G::SPINS_BYTES &&
              a_yp + (K - 1) * ARR + 16 <= (uint32_t)G::SPINS_BYTES && a_ym + (K - 1) * ARR + 16 <= (uint32_t)G::SPINS_BYTES &&
              a_zp + (K - 1) * ARR + 16 <= (uint32_t)G::SPINS_BYTES && a_zm + (K - 1) * ARR + 16 <= (uint32_t)G::SPINS_BYTES);
    RES_CHECK(((a_me | a_x | a_yp | a_ym | a_zp | a_zm) & 15u) == 0u);
    RES_CHECK(KIND == 0 || (fp >= reinterpret_cast<const float4*>(rp.fielda_res) &&
                            fp + (W - 1) * LH < reinterpret_cast<const float4*>(rp.fielda_res) + (size_t)v.D * v.N / 4));
    RES_CHECK(KIND == 1 || (fq >= reinterpret_cast<const uint4*>(rp.fieldb_res) &&
                            fq + (K - 1) * LH < reinterpret_cast<const uint4*>(rp.fieldb_res) + (size_t)v.D * v.N / 16));
    RES_CHECK(!BND || ((!remote_p || rem.off_p + ROWB <= (size_t)v.D * v.Rs * v.N) && (!remote_m || rem.off_m + ROWB <= (size_t)v.D * v.Rs * v.N)));
    RES_CHECK(!BND || (size_t)(ln.ds2 + (uint32_t)c) * (size_t)v.Nh + grow + ROWB <= (size_t)v.D * v.Rs * v.N);
    RES_CHECK(ln.tab_addr >= (uint32_t)__cvta_generic_to_shared(smem + G::SPINS_BYTES) &&
              ln.tab_addr + kResTabBytes <= (uint32_t)__cvta_generic_to_shared(smem + G::SPINS_BYTES) + (uint32_t)rp.cap_reps * kResTabBytes);
    uint4 xr[K];
#pragma unroll
    for (int k = 0; k < K; ++k) xr[k] = *reinterpret_cast<const uint4*>(smem + a_x + k * ARR);
    int r_sn = 0, r_ef = 0, r_hh = 0;                     // measurement partials of the row (MEAS only)
    uint32_t r_ws = 0;
#pragma unroll
    for (int k = 0; k < K; ++k) {             // one 16-site piece of the row at a time
        // field of the piece
        float4 fa[4];
        uint4 fb = make_uint4(0u, 0u, 0u, 0u);
        // Where the field loads stand in program order relative to the piece's shared-memory loads decides how ptxas lays the
        // 128-register loop out: after them is 1.4 % faster in the single-move kernel at L = 64 and a little faster at L = 32,
        // before them 4 % faster in the several-moves-per-launch instantiation at L = 64 (both measured).
        if (!FLATE) {
            if (KIND == 0) fb = __ldg(fq + k * LH);
            else {
#pragma unroll
                for (int w = 0; w < 4; ++w) fa[w] = __ldg(fp + (4 * k + w) * LH);
            }
        }
        ResPiece pc = res_load_piece<K>(smem, xr, a_yp, a_ym, a_zp, a_zm, a_me, k, DIR, rem);
        if (FLATE) {
            if (KIND == 0) fb = __ldg(fq + k * LH);
            else {
#pragma unroll
                for (int w = 0; w < 4; ++w) fa[w] = __ldg(fp + (4 * k + w) * LH);
            }
        }
        const uint32_t fw[4] = {fb.x, fb.y, fb.z, fb.w};
        uint32_t idx8[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) idx8[w] = pc.ns[w] + (pc.me[w] << 3) + (KIND == 0 ? fw[w] : 0u);

        // ---- the four words of the piece ---------------------------------------------------------------
        float mn = 3.0e38f;                   // smallest |d| of the piece (Gaussian)
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const Words4 r = philox_rkreg(rk, q0 + (uint32_t)(4 * k + w), sweep, ln.slot, dom);
            const uint32_t u[4] = {r.w0, r.w1, r.w2, r.w3};
            if (KIND == 0) {
                uint32_t flips = 0;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    // without a zero threshold in the table only the first word of the entry is needed: one wavefront
                    const uint32_t ea = __byte_perm(idx8[w], ln.tab_addr, 0x7650 + j);
                    uint2 ent;
                    if (NEVER) ent = lds64(ea); else { ent.x = lds32(ea); ent.y = 0u; }
                    bool acc = u[j] <= ent.x;
                    if (NEVER) acc = acc && ent.y == 0u;
                    if (acc) flips |= kResSP << (8 * j);
                }
                pc.me[w] ^= flips;
            } else {
                const float a[4] = {fa[w].x, fa[w].y, fa[w].z, fa[w].w};
                float d[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) d[j] = res_gauss_diff(idx8[w], j, ln.tab_addr, a[j], u[j]);
                mn = fminf(fminf(mn, fminf(fabsf(d[0]), fabsf(d[1]))), fminf(fabsf(d[2]), fabsf(d[3])));
                // sign bytes of the four differences -> 0xFF where d < 0 (accept)
                const uint32_t m01 = prmt(__float_as_uint(d[0]), __float_as_uint(d[1]), 0x00FBu);
                const uint32_t m23 = prmt(__float_as_uint(d[2]), __float_as_uint(d[3]), 0xFB00u);
                pc.me[w] ^= prmt(m01, m23, 0x7610u) & (kResSP * 0x01010101u);
            }
        }
        uint4 nw = make_uint4(pc.me[0], pc.me[1], pc.me[2], pc.me[3]);
        if (KIND == 1 && mn < ln.band)          // rare: some site needs the exact binary64 rule
            nw = res_gauss_piece_fix(v, make_uint4(idx8[0], idx8[1], idx8[2], idx8[3]), ln.tab_addr, ln.band, fp + 4 * k * LH, LH,
                                     v.fieldg + ((size_t)(ln.d2 + (uint32_t)c) * (size_t)v.Nh + grow + 16u * k), rr, q0 + 4u * k, sweep, dom);

        // ---- write back ---------------------------------------------------------------------------------
        if (!RAGGED || valid) {
            *reinterpret_cast<uint4*>(smem + a_me + k * ARR) = nw;
            if (BND && (remote_p || remote_m))
                res_piece_to_global(v.spins, (size_t)(ln.ds2 + (uint32_t)c) * (size_t)v.Nh + grow + 16u * k, v.packed, nw);
            if (MEAS) {
                // the final phase (colour 1) measures both colours: its own updated words and the colour-0 words of the same
                // row, xr[k], final since the phase before; their field sits one colour block (L planes x 2 classes) below
                const void* f1 = KIND == 0 ? static_cast<const void*>(fq + k * LH) : static_cast<const void*>(fp + 4 * k * LH);
                const void* f0 = KIND == 0 ? static_cast<const void*>(fq - 2 * G::L * K * LH + k * LH)
                                           : static_cast<const void*>(fp - 2 * G::L * W * LH + 4 * k * LH);
                const int4 m4 = res_measure_piece<KIND>(nw, make_uint4(idx8[0], idx8[1], idx8[2], idx8[3]), xr[k], f1, f0, LH);
                r_sn += m4.x; r_ws += (uint32_t)m4.y; r_ef += m4.z; r_hh += m4.w;
            }
        }
    }
    if (MEAS && (!RAGGED || valid)) {
        // Eb = sum over the colour-1 sites of (2 s - 1)(2 n1 - 6) = 4 s n1 - 12 s - 2 n1 + 6 per site, and summed over a whole
        // (periodic) lattice the n1 of the colour-1 sites count every up spin of colour 0 six times: - 2 sum n1 = - 12 S0.
        // Every plane of a replica ends in the same accumulator, so the row hands in - 12 (its own colour-0 up spins) instead.
        const int S = dot4(r_ws, 0x01010101u) / (int)kResSP;          // up spins of the row, both colours
        m_eb += r_sn / 16 - 12 * S + 6 * ROWB;
        m_ms += 2 * S - 2 * ROWB;
        if (KIND == 0) m_ef += 4 * (r_ef / (int)kResSP) - 2 * r_hh - 2 * S + 2 * ROWB;   // sum (2 hb - 1)(2 s - 1), both colours
        else m_ef += (long long)r_ef * (long long)kResSP;             // SP * (sum of g_i over the up spins), as the accumulators expect
    }
}

// both rows (classes) of a task, one after the other through the same code (the loop body must stay inside the
// instruction cache: two unrolled copies of it were measured 15 % slower)
template <int KIND, int K, bool NEVER, bool UNI, bool BND, bool MEAS, bool RAGGED, bool FLATE = true>
__device__ __forceinline__ void res_task_rows(const View& v, const ResParams& rp, uint8_t* smem, const ResLane& ln, const int c,
                                              const uint32_t sweep, const uint32_t dom, const ResRep* rr, const bool valid,
                                              const bool remote_p, const bool remote_m, const size_t roff_p, const size_t roff_m,
                                              long long& m_eb, long long& m_ef, long long& m_ms) {
#pragma unroll 1
    for (int s = 0; s < 2; ++s)
        res_row<KIND, K, NEVER, UNI, BND, MEAS, RAGGED, FLATE>(v, rp, smem, ln, s, c, (s + c) & 1, sweep, dom, rr, valid, remote_p, remote_m, roff_p, roff_m,
                                                        m_eb, m_ef, m_ms);
}

// K = 16-byte pieces per row per colour (L = 32 K); UNI: one member, round keys come from the constant bank
template <int KIND, int K, bool NEVER, bool UNI, int THREADS, bool MULTI = false>
__global__ void __launch_bounds__(THREADS, 1) k_sweep_res(const View v, const ResParams rp) {
    using G = ResGeom<K>;
    constexpr int L = G::L, LH = G::LH, ROWB = G::ROWB, W = G::W, ARR = G::ARR;
    extern __shared__ __align__(1024) uint8_t smem[];

    const int tid = threadIdx.x, lane = tid & 31;
    const int b = blockIdx.x;
    RES_STAMP(0);
    // the last rp.rem CTAs own one plane more: they hold the hottest replicas, whose planes are slightly cheaper
    // (fewer exact-rule fall-backs), so the longer runs do not also carry the dearer planes
    const int nshort = (int)gridDim.x - rp.rem;                      // CTAs with rp.q planes
    const int start = b * rp.q + max(0, b - nshort);
    const int count = min(rp.q + (b >= nshort ? 1 : 0), rp.total_planes - start);   // (a replica-aligned plan: the last CTA takes what is left)
    if (count <= 0) return;
    const int E = count * LH;                   // rows in use (per colour and class)
    const int nb = (E + 31) / 32;               // 32-row blocks

    uint8_t* s_tab = smem + G::SPINS_BYTES;
    ResRep* s_rep = reinterpret_cast<ResRep*>(s_tab + (size_t)rp.cap_reps * kResTabBytes);
    ResPlane* s_plane = reinterpret_cast<ResPlane*>(s_rep + rp.cap_reps);
    int* s_order = reinterpret_cast<int*>(s_plane + G::MAXPLANES);
    int* s_done = s_order + G::NBCAP;           // per block: tasks completed so far (one per phase)
    int* s_ctl = s_done + G::NBCAP;             // [0],[1] boundary tasks done in the open even / odd phase, [2] next task number, [3] boundary blocks
    long long* s_acc = reinterpret_cast<long long*>(s_ctl + 4);   // [rep][3] measurement accumulators
    long long* s_wacc = s_acc + 3 * rp.cap_reps;                   // [warp][4]: replica held (-1: none), Eb, Ef, Msum of that replica
    // byte offset of row e of array (colour, class, piece)
    auto A = [&](int col, int s, int k, int e) { return (uint32_t)(((col * 2 + s) * K + k) * ARR + e * 16); };

    // ---- set-up: plane table, replica contexts, block order --------------------------------------------
    const int dt0 = start / L;
    const int nrep = (start + count - 1) / L - dt0 + 1;
    for (int p = tid; p < count; p += THREADS) {
        const int P = start + p, dt = P / L, z = P % L;
        const int Pzp = dt * L + (z + 1 == L ? 0 : z + 1), Pzm = dt * L + (z == 0 ? L - 1 : z - 1);
        auto owner = [&](int Q) {
            const int small = nshort * rp.q;
            return Q < small ? Q / rp.q : nshort + (Q - small) / (rp.q + 1);
        };
        ResPlane pi;
        const bool lp = Pzp >= start && Pzp < start + count, lm = Pzm >= start && Pzm < start + count;
        pi.zp_pl = lp ? (int16_t)(Pzp - start) : (int16_t)-1;
        pi.zm_pl = lm ? (int16_t)(Pzm - start) : (int16_t)-1;
        pi.zp_owner = lp ? 0 : (uint8_t)owner(Pzp);
        pi.zm_owner = lm ? 0 : (uint8_t)owner(Pzm);
        pi.rep = (uint8_t)(dt - dt0);
        pi.z = (uint8_t)z;
        s_plane[p] = pi;
    }
    for (int r = tid; r < nrep; r += THREADS) {
        const int dt = dt0 + r, d = rp.d0 + dt / v.n_it, q = dt % v.n_it;
        ResRep rr;
        rr.d = d;
        if (v.shard) { rr.slot = v.stored_slot(q); rr.tr = d * v.R + v.r2t[d * v.R + rr.slot]; }   // visit stored slots
        else { rr.tr = d * v.R + q; rr.slot = v.t2r[rr.tr]; }                                  // visit ranks
        rr.ds = d * v.Rs + v.stored_index(rr.slot);
        rr.band = KIND == 0 ? 0.f : v.band[rr.tr];
        rr.never = KIND == 0 ? v.never[rr.tr] : 0u;
        rr.beta = v.beta[rr.tr];
        uint32_t k0 = v.keys[2 * d], k1 = v.keys[2 * d + 1];
        for (int i = 0; i < 10; ++i) { rr.rk[2 * i] = k0; rr.rk[2 * i + 1] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
        s_rep[r] = rr;
        s_acc[3 * r] = 0; s_acc[3 * r + 1] = 0; s_acc[3 * r + 2] = 0;
    }
    // acceptance tables, 8-byte entries at byte offset SP*n1 + 8*SP*s (+ 16*SP*hb): Gaussian {x, y}, bimodal {thr-1, never}
    for (int i = tid; i < nrep * 32; i += THREADS) {
        const int r = i >> 5, idx = i & 31;
        const int dt = dt0 + r, d = rp.d0 + dt / v.n_it, q = dt % v.n_it;
        const int tr = d * v.R + (v.shard ? v.r2t[d * v.R + v.stored_slot(q)] : q);
        uint2 ent = make_uint2(0u, 0u);
        if (KIND == 0) {
            ent.x = v.etab[(long long)tr * 32 + idx];
            ent.y = (v.never[tr] >> idx) & 1u;
        } else if (idx < 16) {
            const GaussEntry g = v.gtab[(long long)tr * 16 + idx];
            ent.x = __float_as_uint(g.x); ent.y = __float_as_uint(g.y);
        }
        reinterpret_cast<uint2*>(s_tab + (size_t)r * kResTabBytes)[idx] = ent;
    }
    for (int i = tid; i < nb; i += THREADS) s_done[i] = 0;
    if (tid < THREADS / 32) { s_wacc[4 * tid] = -1; s_wacc[4 * tid + 1] = 0; s_wacc[4 * tid + 2] = 0; s_wacc[4 * tid + 3] = 0; }
    if (tid == 0) { s_ctl[0] = 0; s_ctl[1] = 0; s_ctl[2] = 0; s_ctl[3] = 0; }
    __syncthreads();
    // Gaussian Ef = 2 * (sum of g_i over up spins) - (sum of g_i over all sites): the second term, a constant of each plane
    // (ResParams::gsum), goes into the accumulator now, scaled like the first one is measured (SP * sum over up spins)
    if (KIND == 1 && rp.measure && tid < count)
        atomicAdd(reinterpret_cast<unsigned long long*>(s_acc + 3 * s_plane[tid].rep + 1),
                  (unsigned long long)(-(long long)(kResSP / 2) * rp.gsum[(long long)s_rep[s_plane[tid].rep].d * L + s_plane[tid].z]));
    // block order: blocks with a plane whose z-neighbour lives in another CTA first (any order among them)
    {
        bool bnd = false;
        if (tid < nb) {
            const int p0 = (tid * 32) / LH, p1 = min((tid * 32 + 31) / LH, count - 1);
            for (int p = p0; p <= p1; ++p) bnd = bnd || s_plane[p].zp_pl < 0 || s_plane[p].zm_pl < 0;
        }
        if (tid < nb && bnd) s_order[atomicAdd(&s_ctl[3], 1)] = tid;
        __syncthreads();
        const int nbd = s_ctl[3];
        if (tid < nb && !bnd) s_order[nbd + atomicAdd(&s_ctl[0], 1)] = tid;
        __syncthreads();
        if (tid == 0) s_ctl[0] = 0;
    }

    RES_STAMP(1);
    // ---- load the run: global [colour][z][y][ROWB] (0/1) -> shared [colour][s][k][row] (0/SP) ------------------
    // kResLoadDepth loads in flight per thread: the run comes from HBM (or L2) at full rate instead of one
    // round trip per 16-byte piece
    {
        const int units = count * 2 * L * K;            // 16-byte pieces
        for (int u0 = 0; u0 < units; u0 += THREADS * kResLoadDepth) {
            uint4 raw[kResLoadDepth];
            uint32_t dst[kResLoadDepth];
#pragma unroll
            for (int j = 0; j < kResLoadDepth; ++j) {
                const int u = u0 + j * THREADS + tid;
                dst[j] = 0xFFFFFFFFu;
                if (u < units) {
                    const int k = u % K, y = (u / K) % L, col = (u / (K * L)) & 1, p = u / (2 * K * L);
                    const ResPlane pi = s_plane[p];
                    const int ds = s_rep[pi.rep].ds, z = pi.z;
                    RES_CHECK((size_t)(((long long)ds * 2 + col) * v.Nh + ((long long)z * L + y) * ROWB + 16 * k) + 16 <= (size_t)v.D * v.Rs * v.N &&
                              ds >= 0 && ds < v.D * v.Rs && p < count);
                    raw[j] = res_piece_raw(v.spins, (size_t)(((long long)ds * 2 + col) * v.Nh + ((long long)z * L + y) * ROWB + 16 * k), v.packed);
                    dst[j] = A(col, (y + z) & 1, k, p * LH + (y >> 1));
                    RES_CHECK(dst[j] + 16 <= (uint32_t)G::SPINS_BYTES);
                }
            }
#pragma unroll
            for (int j = 0; j < kResLoadDepth; ++j)
                if (dst[j] != 0xFFFFFFFFu) *reinterpret_cast<uint4*>(smem + dst[j]) = res_piece_expand(raw[j], v.packed);
        }
    }
    __syncthreads();
    RES_STAMP(2);
    const int n_bblocks = s_ctl[3];
    const int total_tasks = nb * rp.phases;
    const uint32_t tab0 = (uint32_t)__cvta_generic_to_shared(s_tab);

    // ---- the task flow ------------------------------------------------------------------------------
    constexpr bool RAGGED = (LH % 32) != 0;
    constexpr bool kFieldLate = !(MULTI && K == 2);     // see res_row
    int p_cur = 0, base_cur = 0;                      // phase of this warp's current task number (numbers only grow)
    // MULTI: the launch holds rp.nseg exchange steps; the task flow runs segment by segment (all tasks of the phases up to an
    // exchange step, then a grid-wide rendezvous in which the last CTA to arrive runs the step, then new tables), and a warp
    // that drew a ticket beyond the open segment keeps it for the next one.
    int seg = 0, seg_end = MULTI ? rp.first2 : rp.phases, g_keep = -1;
    for (;;) {
    const int seg_tasks = MULTI ? nb * seg_end : total_tasks;
    for (;;) {
        int g = 0;
        if (MULTI && g_keep >= 0) { g = g_keep; g_keep = -1; }
        else {
            if (lane == 0) g = atomicAdd(&s_ctl[2], 1);
            g = __shfl_sync(0xFFFFFFFFu, g, 0);
        }
        if (g >= seg_tasks) { if (MULTI) g_keep = g; break; }
        while (g - base_cur >= nb) { base_cur += nb; ++p_cur; }
        const int p = p_cur, bidx = g - base_cur;
        const bool meas = rp.measure && p == (MULTI ? seg_end : rp.phases) - 1;   // the last phase before an exchange step (colour 1) also measures, both colours
        const int c = p & 1, oc = 1 - c;
        const uint32_t sweep = rp.sweep0 + (uint32_t)(p >> 1);
        const uint32_t dom = c == 0 ? kDomColour0 : kDomColour1;
        const int eb = s_order[bidx];
        const bool btask = bidx < n_bblocks;
        RES_CHECK(eb >= 0 && eb < nb && p >= 0 && p < rp.phases && lds_volatile(s_done + eb) <= p);
        const int e_raw = eb * 32 + lane;
        const bool valid = !RAGGED || e_raw < E;
        const int e = valid ? e_raw : E - 1;
        const int pl = (int)((unsigned)e / (unsigned)LH), i = (int)((unsigned)e % (unsigned)LH);
        const ResPlane pi = s_plane[pl];
        const ResRep* rr = s_rep + pi.rep;
        const int z = pi.z;
        RES_CHECK(pl >= 0 && pl < count && (int)pi.rep < nrep && z < L && (int)pi.zp_pl < count && (int)pi.zm_pl < count);
        RES_CHECK((pi.zp_pl >= 0 || (int)pi.zp_owner < (int)gridDim.x) && (pi.zm_pl >= 0 || (int)pi.zm_owner < (int)gridDim.x));
        const bool remote_p = pi.zp_pl < 0, remote_m = pi.zm_pl < 0;
        const int e_zp = remote_p ? 0 : pi.zp_pl * LH + i, e_zm = remote_m ? 0 : pi.zm_pl * LH + i;

        // dependencies: the blocks of my plane and of its z-neighbours have finished phase p-1;
        // remote neighbour planes: their owners have published phase p-1
        if (p > 0) {
            const int b_zp = remote_p ? eb : e_zp >> 5, b_zm = remote_m ? eb : e_zm >> 5;
            const int d0 = lds_acquire(s_done + eb), d1 = lds_acquire(s_done + b_zp), d2 = lds_acquire(s_done + b_zm);
            const bool ok = min(d0, min(d1, d2)) >= p;
            if (btask || !__all_sync(0xFFFFFFFFu, ok))
                res_wait_slow(s_done, eb, b_zp, b_zm, p, remote_p ? rp.prog + pi.zp_owner : nullptr,
                              remote_m ? rp.prog + pi.zm_owner : nullptr, (rp.epoch << 8) | (uint32_t)p, rp.diag);
        }

        // per-task lane constants; everything class-dependent is an immediate offset from these
        ResLane ln;
        {
            const uint32_t e16 = (uint32_t)e * 16u, p16 = (uint32_t)(e - i) * 16u;      // my row / first row of my plane
            const uint32_t base_c = (uint32_t)(c * 2 * K) * ARR, base_oc = (uint32_t)(oc * 2 * K) * ARR;
            ln.me = base_c + e16; ln.x = base_oc + e16;
            ln.ya = base_oc + p16 + (uint32_t)((i + 1) & (LH - 1)) * 16u;
            ln.yb = ln.x;
            ln.yc = base_oc + p16 + (uint32_t)((i - 1) & (LH - 1)) * 16u;
            ln.zp = base_oc + (uint32_t)e_zp * 16u; ln.zm = base_oc + (uint32_t)e_zm * 16u;
            ln.q00 = (uint32_t)W * (uint32_t)(2 * i + L * z);
            ln.slot = (uint32_t)rr->slot;
            ln.tab_addr = tab0 + (uint32_t)pi.rep * kResTabBytes;
            ln.band = rr->band;
            ln.zpar = (uint32_t)z & 1u;
            ln.ds2 = (uint32_t)rr->ds * 2u; ln.d2 = (uint32_t)rr->d * 2u;
            const uint32_t fblk0 = ((ln.d2 + (uint32_t)c) * L + (uint32_t)z) * 2u;        // field block of (colour, plane, class 0)
            ln.fp0 = reinterpret_cast<const float4*>(rp.fielda_res) + (size_t)(fblk0 * (W * LH) + (uint32_t)i);
            ln.fq0 = reinterpret_cast<const uint4*>(rp.fieldb_res) + (size_t)(fblk0 * (K * LH) + (uint32_t)i);
            ln.grow0 = (uint32_t)(z * L + 2 * i) * ROWB;
        }

        long long m_eb = 0, m_ef = 0, m_ms = 0;
        if (!btask && !meas) {
            res_task_rows<KIND, K, NEVER, UNI, false, false, RAGGED, kFieldLate>(v, rp, smem, ln, c, sweep, dom, rr, valid, false, false, 0u, 0u, m_eb, m_ef, m_ms);
        } else {
            // rows of a z-neighbour plane that lives in another CTA: read from global memory (class 0; class 1 = + ROWB)
            const int zq_p = (z + 1) & (L - 1), zq_m = (z - 1) & (L - 1);
            const size_t roff_p = (size_t)(ln.ds2 + (uint32_t)oc) * (size_t)v.Nh + (uint32_t)(zq_p * L + 2 * i) * ROWB;
            const size_t roff_m = (size_t)(ln.ds2 + (uint32_t)oc) * (size_t)v.Nh + (uint32_t)(zq_m * L + 2 * i) * ROWB;
            if (btask && !meas)
                res_task_rows<KIND, K, NEVER, UNI, true, false, RAGGED, kFieldLate>(v, rp, smem, ln, c, sweep, dom, rr, valid, remote_p, remote_m, roff_p, roff_m, m_eb, m_ef, m_ms);
            else
                res_task_rows<KIND, K, NEVER, UNI, true, true, RAGGED, kFieldLate>(v, rp, smem, ln, c, sweep, dom, rr, valid, remote_p && btask, remote_m && btask, roff_p, roff_m, m_eb, m_ef, m_ms);
        }

        if (meas) {
            // per-replica sums: a warp keeps the sums of the replica it is working on in its own shared-memory slot (plain
            // read-modify-write by lane 0) and hands them to the CTA's accumulators only when the replica changes and after
            // its last task: the 64-bit shared-memory atomics (compare-and-swap loops) would otherwise all collide at the
            // end of the measuring phase.  A warp that straddles a replica seam adds lane by lane.
            const int rep = valid ? (int)pi.rep : -1;
            const int rep0 = __shfl_sync(0xFFFFFFFFu, rep, 0);
            if (__all_sync(0xFFFFFFFFu, rep == rep0 || rep < 0)) {
                m_eb = warp_sum(m_eb); m_ef = warp_sum(m_ef); m_ms = warp_sum(m_ms);
                if (lane == 0 && rep0 >= 0) {
                    long long* wa = s_wacc + 4 * (tid >> 5);
                    if (wa[0] != (long long)rep0) {
                        res_flush_sums(s_acc, (int)wa[0], wa[1], wa[2], wa[3]);
                        wa[0] = rep0; wa[1] = 0; wa[2] = 0; wa[3] = 0;
                    }
                    wa[1] += m_eb; wa[2] += m_ef; wa[3] += m_ms;
                }
            } else {
                res_flush_sums(s_acc, rep, m_eb, m_ef, m_ms);
            }
        }
        __syncwarp();
        if (lane == 0) {
            if (btask) {
                // a neighbour CTA only needs phase p+1 of mine after it has seen phase p published, and it publishes
                // its own phase p+1 only after that: at most two phases are open at once, one counter per parity
                __threadfence();
                const int done = atomicAdd(&s_ctl[p & 1], 1) + 1;
                if (done == n_bblocks) {
                    atomicExch(&s_ctl[p & 1], 0);
                    __threadfence();
                    st_release_gpu(rp.prog + b, (rp.epoch << 8) | (uint32_t)(p + 1));
                }
            }
            sts_release_inc(&s_done[eb]);
        }
    }
    if (!MULTI || seg == rp.nseg - 1) break;
    // ---- an exchange step inside the launch (MULTI) ------------------------------------------------------------
    {
        if (lane == 0) {
            long long* wa = s_wacc + 4 * (tid >> 5);
            res_flush_sums(s_acc, (int)wa[0], wa[1], wa[2], wa[3]);
            wa[0] = -1; wa[1] = 0; wa[2] = 0; wa[3] = 0;
        }
        __syncthreads();
        for (int r = tid; r < nrep * 3; r += THREADS) {
            const long long val = (KIND == 1 && r % 3 == 1) ? s_acc[r] / (long long)(kResSP / 2) : s_acc[r];
            atomicAdd(reinterpret_cast<unsigned long long*>(v.acc + (long long)(s_rep[r / 3].d * v.R + s_rep[r / 3].slot) * 3 + r % 3), (unsigned long long)val);
        }
        __threadfence();
        __syncthreads();
        if (tid == 0) s_ctl[0] = (atomicAdd(rp.ticket, 1u) == (uint32_t)(rp.nact * (seg + 1) - 1)) ? 1 : 0;   // (no boundary task is open: the slot is free)
        __syncthreads();
        const uint32_t xwant = (rp.epoch << 8) | (uint32_t)(seg + 1);
        if (s_ctl[0]) {                                // every CTA's sums are in View::acc: this one runs the step
            __threadfence();
            for (int d = 0; d < v.D; ++d) {
                exchange_member(v, d, rp.xstep + (uint32_t)seg, rp.xrow + seg, 1);
                __syncthreads();
            }
            __threadfence();
            if (tid == 0) st_release_gpu(rp.xflag, xwant);
        } else if (tid == 0) {
            int polls = 0;
            while (ld_acquire_gpu(rp.xflag) != xwant) {
                backoff();
                if (++polls > (1 << 22)) { atomicOr(rp.diag, 1ull); break; }
            }
        }
        __syncthreads();
        if (tid == 0) s_ctl[0] = 0;
        // the resident lattices keep their slots; their ranks (temperatures) are the new ones
        for (int r = tid; r < nrep; r += THREADS) {
            const int d = s_rep[r].d, tr = d * v.R + __ldcg(v.r2t + d * v.R + s_rep[r].slot);
            s_rep[r].tr = tr;
            s_rep[r].band = KIND == 0 ? 0.f : v.band[tr];
            s_rep[r].never = KIND == 0 ? v.never[tr] : 0u;
            s_rep[r].beta = v.beta[tr];
            s_acc[3 * r] = 0; s_acc[3 * r + 1] = 0; s_acc[3 * r + 2] = 0;
        }
        for (int i = tid; i < nrep * 32; i += THREADS) {
            const int r = i >> 5, idx = i & 31;
            const int d = s_rep[r].d, tr = d * v.R + __ldcg(v.r2t + d * v.R + s_rep[r].slot);
            uint2 ent = make_uint2(0u, 0u);
            if (KIND == 0) {
                ent.x = v.etab[(long long)tr * 32 + idx];
                ent.y = (v.never[tr] >> idx) & 1u;
            } else if (idx < 16) {
                const GaussEntry ge = v.gtab[(long long)tr * 16 + idx];
                ent.x = __float_as_uint(ge.x); ent.y = __float_as_uint(ge.y);
            }
            reinterpret_cast<uint2*>(s_tab + (size_t)r * kResTabBytes)[idx] = ent;
        }
        __syncthreads();
        if (KIND == 1 && tid < count)
            atomicAdd(reinterpret_cast<unsigned long long*>(s_acc + 3 * s_plane[tid].rep + 1),
                      (unsigned long long)(-(long long)(kResSP / 2) * rp.gsum[(long long)s_rep[s_plane[tid].rep].d * L + s_plane[tid].z]));
        __syncthreads();
        ++seg;
        seg_end += rp.period2;
    }
    }
    if (lane == 0) {                                  // hand this warp's measurement sums over
        long long* wa = s_wacc + 4 * (tid >> 5);
        res_flush_sums(s_acc, (int)wa[0], wa[1], wa[2], wa[3]);
    }
    RES_STAMP(3);
    __syncthreads();
    RES_STAMP(4);

    // ---- store the run back, hand the measurement over ------------------------------------------------------
    {
        const int units = count * 2 * L * K;
        for (int u = tid; u < units; u += THREADS) {
            const int k = u % K, y = (u / K) % L, col = (u / (K * L)) & 1, p = u / (2 * K * L);
            const ResPlane pi = s_plane[p];
            const int ds = s_rep[pi.rep].ds, z = pi.z;
            const uint4 x = *reinterpret_cast<const uint4*>(smem + A(col, (y + z) & 1, k, p * LH + (y >> 1)));
            res_piece_to_global(v.spins, (size_t)(((long long)ds * 2 + col) * v.Nh + ((long long)z * L + y) * ROWB + 16 * k), v.packed, x);
        }
        if (rp.measure)
            for (int r = tid; r < nrep * 3; r += THREADS)
            {
                // Gaussian Ef: the accumulator holds SP * (sum of g_i over up spins) - (SP / 2) * (sum of g_i over the planes held)
                const long long val = (KIND == 1 && r % 3 == 1) ? s_acc[r] / (long long)(kResSP / 2) : s_acc[r];
                atomicAdd(reinterpret_cast<unsigned long long*>(v.acc + (long long)(s_rep[r / 3].d * v.R + s_rep[r / 3].slot) * 3 + r % 3), (unsigned long long)val);
            }
    }
    RES_STAMP(5);
    if (rp.exchange) {
        // the CTA that arrives last has every replica's sums in View::acc (integer atomics at L2): it runs the exchange step
        __threadfence();
        __syncthreads();
        if (tid == 0) s_ctl[0] = (atomicAdd(rp.ticket, 1u) == (uint32_t)(rp.nact * (MULTI ? rp.nseg : 1) - 1)) ? 1 : 0;
        __syncthreads();
        if (s_ctl[0]) {
            __threadfence();
            for (int d = 0; d < v.D; ++d) {
                exchange_member(v, d, rp.xstep + (MULTI ? (uint32_t)(rp.nseg - 1) : 0u), rp.xrow + (MULTI ? rp.nseg - 1 : 0), 1);
                __syncthreads();
            }
            if (tid == 0) *rp.ticket = 0u;
        }
    }
    RES_STAMP(6);
}

}  // namespace rfim
