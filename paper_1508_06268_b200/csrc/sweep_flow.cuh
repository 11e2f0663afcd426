// sweep_flow.cuh -- the tuned sweep: one persistent launch covers every phase (colour 0 / colour 1 of
// each sweep) of a whole exchange period, for every replica.  DESIGN.md section 6.
//
// Work item = (phase p, member d, replica group g, z-slab sl).  Items are numbered phase-major and
// dealt round-robin to the co-resident CTAs (cooperative launch).  An item of phase p may start as
// soon as the three slabs sl-1, sl, sl+1 of its own replica group have finished phase p-1 (a
// per-(group,slab) progress word in global memory, release/acquire at gpu scope): no grid-wide
// barrier, no per-colour launch, CTAs flow from one phase into the next.
//
// Inside an item a CTA of 256 threads owns 256*CPT chunks (16 same-colour sites = one uint4 = four
// Philox calls each).  The chunk position is fixed for all replicas of the group, so the disorder
// field of those sites is loaded into registers once per item and reused RR times.  The other
// colour's ZT+2 planes are staged in shared memory with cp.async (L2 -> smem, bypassing the
// incoherent L1); the six neighbour words of a chunk are then five LDS.128 plus, for L = 64, one LDS.32.
#pragma once
#include <cstdint>
#include <cstring>
#include "kernels_ref.cuh"
#include "philox.cuh"
#include "view.h"

namespace rfim {

constexpr int kFlowThreads = 256;
constexpr int kFlowMaxMembers = 32;

struct FlowParams {
    int RR, G;                       // replicas per group, groups per member
    int d0, nd;                      // members [d0, d0+nd) are covered by this launch
    int phases;                      // 2 * sweeps of this launch, <= 254
    uint32_t sweep0;                 // global sweep index of phase 0
    uint32_t epoch;                  // launch id: progress words hold (epoch << 8) | phases done
    uint32_t* prog;                  // [D][R][S] progress words (indexed [d][g][sl], g < G <= R)
    int prog_stride_d, prog_stride_g;
    unsigned long long* diag;        // diag[0] |= 1 if a dependency wait timed out (results invalid, no hang)
    uint32_t rk[kFlowMaxMembers][20];  // Philox round keys per member: rk[2r] = k0 + r*W0, rk[2r+1] = k1 + r*W1
};

// ---- small device helpers ----------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
#if defined(__CUDA_ARCH__)
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gsrc) : "memory");
#else
    memcpy(smem_dst, gsrc, 16);
#endif
}
__device__ __forceinline__ void cp_async_wait_all() {
#if defined(__CUDA_ARCH__)
    asm volatile("cp.async.wait_all;" ::: "memory");
#endif
}
__device__ __forceinline__ uint32_t ld_acquire_gpu(const uint32_t* p) {
#if defined(__CUDA_ARCH__)
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
#else
    return *p;
#endif
}
__device__ __forceinline__ void st_release_gpu(uint32_t* p, uint32_t v) {
#if defined(__CUDA_ARCH__)
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
#else
    *p = v;
#endif
}
__device__ __forceinline__ uint4 ld_cg16(const void* p) {
#if defined(__CUDA_ARCH__)
    return __ldcg(reinterpret_cast<const uint4*>(p));
#else
    return *reinterpret_cast<const uint4*>(p);
#endif
}
__device__ __forceinline__ void backoff() {
#if defined(__CUDA_ARCH__)
    __nanosleep(64);
#endif
}

// Philox4x32-10 with the key schedule supplied (warp-uniform, from kernel parameters)
__device__ __forceinline__ Words4 philox_rk(const uint32_t* __restrict__ rk, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
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

struct ReplicaCtx {        // per-replica values every thread of the CTA needs (shared memory)
    int slot;
    uint32_t never;
    float band;
    double beta;
};

// exact rule for the four sites of one word (rare: taken when any of them fell inside the guard band)
__device__ __noinline__ uint32_t gauss_word_exact(const View& v, uint32_t me, uint32_t sum, const int32_t* __restrict__ g4, double beta,
                                                  uint32_t u0, uint32_t u1, uint32_t u2, uint32_t u3) {
    uint32_t flips = 0;
    const uint32_t u[4] = {u0, u1, u2, u3};
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (gauss_accept_exact(v, (int)((me >> (8 * k)) & 1u), (int)((sum >> (8 * k)) & 0xFFu), g4[k], beta, u[k])) flips |= 1u << (8 * k);
    return flips;
}

// Update the 16 sites of one chunk.  me/c/yp/ym/zp/zm: own word and the five aligned neighbour words (x4);
// adj: the word holding the far x-neighbour of the chunk's edge byte (C == 2), PAR: x-parity of the row.
template <int KIND, int C, int PAR, bool NEVER>
__device__ __forceinline__ uint4 update_chunk16(const View& v, const uint4 me4, const uint4 c4, const uint4 yp, const uint4 ym,
                                                const uint4 zp, const uint4 zm, const uint32_t adj, const float* __restrict__ a,
                                                const uint4 fb, const void* __restrict__ tab, const ReplicaCtx& rc,
                                                const uint32_t* __restrict__ rk, uint32_t word0, uint32_t sweep, uint32_t dom,
                                                const int32_t* __restrict__ gchunk) {
    const uint32_t me[4] = {me4.x, me4.y, me4.z, me4.w};
    const uint32_t cw[4] = {c4.x, c4.y, c4.z, c4.w};
    const uint32_t a1[4] = {yp.x + ym.x, yp.y + ym.y, yp.z + ym.z, yp.w + ym.w};
    const uint32_t a2[4] = {zp.x + zm.x, zp.y + zm.y, zp.z + zm.z, zp.w + zm.w};
    const uint32_t fw[4] = {fb.x, fb.y, fb.z, fb.w};
    uint32_t out[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint32_t sh;
        if (PAR == 0) {
            const uint32_t prev = (i == 0) ? (C == 1 ? cw[3] : adj) : cw[i - 1];
            sh = __funnelshift_r(prev, cw[i], 24);           // byte k <- other[xh - 1]
        } else {
            const uint32_t next = (i == 3) ? (C == 1 ? cw[0] : adj) : cw[i + 1];
            sh = __funnelshift_r(cw[i], next, 8);            // byte k <- other[xh + 1]
        }
        const uint32_t sum = cw[i] + sh + a1[i] + a2[i];     // per byte: number of up neighbours, 0..6
        const Words4 r = philox_rk(rk, word0 + (uint32_t)i, sweep, (uint32_t)rc.slot, dom);
        const uint32_t u[4] = {r.w0, r.w1, r.w2, r.w3};
        uint32_t flips = 0;
        if (KIND == 0) {
            const uint32_t idxw = sum + (me[i] << 3) + fw[i];           // n1 | s<<3 | hb<<4 per byte
            const uint32_t* et = reinterpret_cast<const uint32_t*>(tab);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t idx = __byte_perm(idxw, 0u, 0x4440u + k);
                bool acc = u[k] <= et[idx];
                if (NEVER) acc = acc && !((rc.never >> idx) & 1u);
                if (acc) flips |= 1u << (8 * k);
            }
        } else {
            const uint32_t idxw = sum + (me[i] << 3);                   // n1 | s<<3 per byte
            const GaussEntry* gt = reinterpret_cast<const GaussEntry*>(tab);
            bool amb = false;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t idx = __byte_perm(idxw, 0u, 0x4440u + k);
                const GaussEntry e = gt[idx];
                const float P = ex2_approx(fmaf(a[4 * i + k], e.y, e.x));
                const float d = __uint2float_rn(u[k]) - P;
                amb = amb || (fabsf(d) < rc.band);
                if (d < 0.0f) flips |= 1u << (8 * k);
            }
            if (amb) flips = gauss_word_exact(v, me[i], sum, gchunk + 4 * i, rc.beta, u[0], u[1], u[2], u[3]);
        }
        out[i] = me[i] ^ flips;
    }
    return make_uint4(out[0], out[1], out[2], out[3]);
}

// C = chunks per row per colour (L = 32*C), CPT = chunks per thread, ZT = planes per slab = 256*CPT/(L*C)
template <int KIND, int C, int CPT, bool NEVER>
__global__ void __launch_bounds__(kFlowThreads) k_sweep_flow(const View v, const FlowParams fp) {
    constexpr int L = 32 * C;
    constexpr int ROWB = 16 * C;                 // bytes per row per colour
    constexpr int PLANEB = L * ROWB;             // bytes per plane per colour
    constexpr int ZT = kFlowThreads * CPT / (L * C);
    constexpr int S = L / ZT;
    constexpr int HALF = ZT * (L / 2) * C;       // chunk slots per x-parity class
    constexpr int STAGE_GRANULES = (ZT + 2) * L * C;
    static_assert(ZT * L * C == kFlowThreads * CPT && S >= 3, "tile shape");

    __shared__ uint4 s_stage[STAGE_GRANULES];                     // other colour, planes z0-1 .. z0+ZT
    __shared__ uint2 s_tab[16];                                   // this replica's table (Gaussian 16 x 8 B; bimodal 32 x 4 B)
    __shared__ ReplicaCtx s_rc;

    const int tid = threadIdx.x;
    const long long Nh = v.Nh;
    const long long per_phase = (long long)fp.nd * fp.G * S;
    const long long total = per_phase * fp.phases;

    for (long long it = blockIdx.x; it < total; it += gridDim.x) {
        const int p = (int)(it / per_phase);
        const int rem = (int)(it % per_phase);
        const int dl = rem / (fp.G * S);
        const int g = (rem / S) % fp.G;
        const int sl = rem % S;
        const int d = fp.d0 + dl;
        const int colour = p & 1;
        const uint32_t sweep = fp.sweep0 + (uint32_t)(p >> 1);
        const uint32_t dom = colour == 0 ? kDomColour0 : kDomColour1;
        const int z0 = sl * ZT;
        const uint32_t* rk = fp.rk[dl];
        uint32_t* prog = fp.prog + (long long)d * fp.prog_stride_d + (long long)g * fp.prog_stride_g;

        // ---- chunk geometry and field registers: fixed for every replica of the group -----------------
        int o_c[CPT], o_yp[CPT], o_ym[CPT], o_adj[CPT], par[CPT];
        long long go[CPT];                               // byte offset of the chunk inside a colour array
        float a[CPT][16];
        uint4 fb[CPT];
#pragma unroll
        for (int ci = 0; ci < CPT; ++ci) {
            const int s = tid + kFlowThreads * ci;
            const int P = (HALF == kFlowThreads) ? ci : s / HALF;
            const int r1 = s % HALF;
            const int zl = r1 / ((L / 2) * C);
            const int e = (r1 / C) % (L / 2);
            const int cx = r1 % C;
            const int z = z0 + zl;
            const int y = 2 * e + ((P + z + colour) & 1);
            const int yp = (y + 1) & (L - 1), ym = (y - 1) & (L - 1);
            par[ci] = P;
            o_c[ci] = ((zl + 1) * L + y) * ROWB + 16 * cx;
            o_yp[ci] = ((zl + 1) * L + yp) * ROWB + 16 * cx;
            o_ym[ci] = ((zl + 1) * L + ym) * ROWB + 16 * cx;
            o_adj[ci] = ((zl + 1) * L + y) * ROWB + 16 * (1 - cx) + (P == 0 ? 12 : 0);
            go[ci] = ((long long)z * L + y) * ROWB + 16 * cx;
            const long long fo = ((long long)d * 2 + colour) * Nh + go[ci];
            if (KIND == 0) {
                fb[ci] = *reinterpret_cast<const uint4*>(v.fieldb + fo);
            } else {
                fb[ci] = make_uint4(0, 0, 0, 0);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 f = *reinterpret_cast<const float4*>(v.fielda + fo + 4 * q);
                    a[ci][4 * q + 0] = f.x; a[ci][4 * q + 1] = f.y; a[ci][4 * q + 2] = f.z; a[ci][4 * q + 3] = f.w;
                }
            }
        }

        // ---- dependencies: slabs sl-1, sl, sl+1 of this group must have finished phase p-1 ------------
        if (p > 0 && tid < 3) {
            const uint32_t want = (fp.epoch << 8) | (uint32_t)p;
            const uint32_t* w = prog + ((sl + tid - 1 + S) % S);
            int spins = 0;
            while ((int32_t)(ld_acquire_gpu(w) - want) < 0) {
                backoff();
                if (++spins > (1 << 22)) { atomicOr(fp.diag, 1ull); break; }
            }
        }
        __syncthreads();

        for (int rr = 0; rr < fp.RR; ++rr) {
            const int t = g * fp.RR + rr;
            if (t >= v.n) break;
            const int tr = d * v.R + t;
            const int slot = v.t2r[tr];
            uint8_t* mine = v.spins + ((long long)(d * v.R + slot) * 2 + colour) * Nh;
            const uint8_t* other = v.spins + ((long long)(d * v.R + slot) * 2 + (1 - colour)) * Nh;

            // stage the other colour's planes z0-1 .. z0+ZT (periodic) and this rank's table
            for (int gi = tid; gi < STAGE_GRANULES; gi += kFlowThreads) {
                const int zz = gi / (L * C);
                const int z = (z0 - 1 + zz + L) & (L - 1);
                cp_async16(&s_stage[gi], other + (long long)z * PLANEB + (long long)(gi % (L * C)) * 16);
            }
            if (tid < 16) {
                if (KIND == 0) s_tab[tid] = reinterpret_cast<const uint2*>(v.etab + (long long)tr * 32)[tid];
                else s_tab[tid] = reinterpret_cast<const uint2*>(v.gtab + (long long)tr * 16)[tid];
            }
            if (tid == 32) {
                s_rc.slot = slot;
                s_rc.never = KIND == 0 ? v.never[tr] : 0u;
                s_rc.band = KIND == 0 ? 0.f : v.band[tr];
                s_rc.beta = v.beta[tr];
            }
            uint4 me[CPT];
#pragma unroll
            for (int ci = 0; ci < CPT; ++ci) me[ci] = ld_cg16(mine + go[ci]);
            cp_async_wait_all();
            __syncthreads();

            const ReplicaCtx rc = s_rc;
            const uint8_t* st = reinterpret_cast<const uint8_t*>(s_stage);
#pragma unroll
            for (int ci = 0; ci < CPT; ++ci) {
                const uint4 c4 = *reinterpret_cast<const uint4*>(st + o_c[ci]);
                const uint4 yp = *reinterpret_cast<const uint4*>(st + o_yp[ci]);
                const uint4 ym = *reinterpret_cast<const uint4*>(st + o_ym[ci]);
                const uint4 zp = *reinterpret_cast<const uint4*>(st + o_c[ci] + PLANEB);
                const uint4 zm = *reinterpret_cast<const uint4*>(st + o_c[ci] - PLANEB);
                const uint32_t adj = (C == 1) ? 0u : *reinterpret_cast<const uint32_t*>(st + o_adj[ci]);
                const uint32_t word0 = (uint32_t)(go[ci] >> 2);
                const int32_t* gchunk = KIND == 0 ? nullptr : v.fieldg + ((long long)d * 2 + colour) * Nh + go[ci];
                uint4 nw;
                if (par[ci] == 0)
                    nw = update_chunk16<KIND, C, 0, NEVER>(v, me[ci], c4, yp, ym, zp, zm, adj, a[ci], fb[ci], s_tab, rc, rk, word0, sweep, dom, gchunk);
                else
                    nw = update_chunk16<KIND, C, 1, NEVER>(v, me[ci], c4, yp, ym, zp, zm, adj, a[ci], fb[ci], s_tab, rc, rk, word0, sweep, dom, gchunk);
                *reinterpret_cast<uint4*>(mine + go[ci]) = nw;
            }
            __syncthreads();             // everyone is done with s_stage / s_tab / s_rc
        }

        // ---- publish: this slab of this group has finished phase p --------------------------------------
        __threadfence();
        __syncthreads();
        if (tid == 0) st_release_gpu(prog + sl, (fp.epoch << 8) | (uint32_t)(p + 1));
    }
}

// ---- fast energy / magnetisation reduction: one thread per word of colour 0 (L % 8 == 0) --------------------
// Eb = sum over colour-0 sites of s_i * (six-neighbour sum) (every bond has exactly one colour-0 end).
__device__ __forceinline__ int dot4(uint32_t a, uint32_t b) {
#if defined(__CUDA_ARCH__)
    return (int)__dp4a(a, b, 0u);
#else
    int s = 0;
    for (int k = 0; k < 4; ++k) s += (int)((a >> (8 * k)) & 0xFFu) * (int)((b >> (8 * k)) & 0xFFu);
    return s;
#endif
}

__global__ void k_reduce_word(View v) {
    const int d = blockIdx.y / v.n, t = blockIdx.y % v.n;
    const int slot = v.t2r[d * v.R + t];
    const int NW = (int)(v.Nh >> 2);
    if (!v.stores(slot)) return;                                              // a replica shard reduces the slots it stores
    const uint32_t* c0 = reinterpret_cast<const uint32_t*>(v.spins + (long long)(d * v.Rs + v.stored_index(slot)) * 2 * v.Nh);
    const uint32_t* c1 = c0 + NW;
    const long long f0 = (long long)d * 2 * v.Nh;
    const int L = v.L, W = v.W;
    long long eb = 0, ef = 0, ms = 0;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < NW; q += gridDim.x * blockDim.x) {
        const int w = q % W;
        const int y = (q / W) % L;
        const int z = q / (W * L);
        const int par = (y + z) & 1;
        const int yp = y + 1 == L ? 0 : y + 1, ym = y == 0 ? L - 1 : y - 1;
        const int zp = z + 1 == L ? 0 : z + 1, zm = z == 0 ? L - 1 : z - 1;
        const int row = W * (y + L * z);
        const uint32_t c = c1[row + w];
        uint32_t sh;
        if (par == 0) sh = __funnelshift_r(c1[row + (w == 0 ? W - 1 : w - 1)], c, 24);
        else sh = __funnelshift_r(c, c1[row + (w + 1 == W ? 0 : w + 1)], 8);
        const uint32_t sum = c + sh + c1[W * (yp + L * z) + w] + c1[W * (ym + L * z) + w] + c1[W * (y + L * zp) + w] + c1[W * (y + L * zm) + w];
        const uint32_t s0 = c0[q];
        // sum over the word of (2 s - 1)(2 n1 - 6) = 4 s.n1 - 12 s - 2 n1 + 6
        const int sn = dot4(s0, sum), ss = dot4(s0, 0x01010101u), nn = dot4(sum, 0x01010101u), s1s = dot4(c, 0x01010101u);
        eb += 4 * sn - 12 * ss - 2 * nn + 24;
        ms += 2 * (ss + s1s) - 8;
        if (v.kind == 0) {
            const uint32_t h0 = *reinterpret_cast<const uint32_t*>(v.fieldb + f0 + 4 * q) >> 4;             // 0/1 per byte
            const uint32_t h1 = *reinterpret_cast<const uint32_t*>(v.fieldb + f0 + v.Nh + 4 * q) >> 4;
            // sum (2h-1)(2s-1) = 4 h.s - 2 h - 2 s + 1 per site
            ef += 4 * dot4(h0, s0) - 2 * dot4(h0, 0x01010101u) - 2 * ss + 4;
            ef += 4 * dot4(h1, c) - 2 * dot4(h1, 0x01010101u) - 2 * s1s + 4;
        } else {
            const int4 g0 = *reinterpret_cast<const int4*>(v.fieldg + f0 + 4 * q);
            const int4 g1 = *reinterpret_cast<const int4*>(v.fieldg + f0 + v.Nh + 4 * q);
            const int gg0[4] = {g0.x, g0.y, g0.z, g0.w}, gg1[4] = {g1.x, g1.y, g1.z, g1.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                ef += ((s0 >> (8 * k)) & 1u) ? (long long)gg0[k] : -(long long)gg0[k];
                ef += ((c >> (8 * k)) & 1u) ? (long long)gg1[k] : -(long long)gg1[k];
            }
        }
    }
    eb = warp_sum(eb); ef = warp_sum(ef); ms = warp_sum(ms);
    if ((threadIdx.x & 31) == 0) {
        long long* acc = v.acc + (long long)(d * v.R + slot) * 3;
        atomicAdd(reinterpret_cast<unsigned long long*>(acc + 0), (unsigned long long)eb);
        atomicAdd(reinterpret_cast<unsigned long long*>(acc + 1), (unsigned long long)ef);
        atomicAdd(reinterpret_cast<unsigned long long*>(acc + 2), (unsigned long long)ms);
    }
}

}  // namespace rfim
