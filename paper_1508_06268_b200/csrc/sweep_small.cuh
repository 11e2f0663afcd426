// sweep_small.cuh -- small lattices (L = 8, 16, ...: L % 8 == 0, the whole lattice of a replica fits in shared
// memory, and the plane-run kernel of sweep_res.cuh does not apply): one CTA per replica keeps BOTH colours of the
// lattice in shared memory for a whole exchange period.  One launch = k sweeps (2k phases separated by a block
// barrier) + the per-replica energy / magnetisation reduction + the exchange step (run by the CTA that finishes last),
// i.e. one launch per parallel-tempering move instead of 2k + 2 (the paper's own sizes are
// L = 8, 16, 32, 64; its kernel needs two launches per sweep).  DESIGN.md section 6.
//
// The arithmetic is that of the one-launch-per-colour word kernel (kernels_ref.cuh): a thread owns 32-bit words of
// four same-colour sites = one Philox call, neighbour counts are byte-wise sums of the other colour's words, the
// acceptance goes through bimodal_accept / gauss_accept (float path with guard band, exact binary64 rule inside it).
#pragma once
#include <cstdint>
#include "kernels_ref.cuh"
#include "philox.cuh"
#include "sweep_flow.cuh"
#include "view.h"

namespace rfim {

constexpr int kSmallMaxThreads = 1024;

struct SmallParams {
    int phases;                  // 2 * sweeps of this launch
    int measure;                 // != 0: reduce (Eb, Ef, Msum) of every replica into View::acc after the last phase
    int exchange;                // != 0: the CTA that finishes last runs the exchange step of every member
    uint32_t xstep;              // exchange step index, time-series row (exchange != 0)
    long long xrow;
    uint32_t* ticket;            // arrival counter (left at zero)
    uint32_t sweep0;             // global sweep index of phase 0
    // several parallel-tempering moves per launch (cooperative launches only): the launch ends on an exchange step and holds nseg
    // of them, after phase first2 - 1, first2 + period2 - 1, ...; the lattices stay in shared memory across them
    int nseg, first2, period2;
    uint32_t* xflag;             // release word of the mid-launch exchange steps: (epoch << 8) | steps done
    uint32_t epoch;
    unsigned long long* diag;
};

__host__ __device__ inline size_t small_smem_bytes(long long N) { return (size_t)N + 32 * 8 + 3 * 32 * sizeof(long long); }

// six-neighbour byte sums of word (w, y, z) of colour c from the other colour's words `o` (shared memory)
__device__ __forceinline__ uint32_t small_neighbours(const uint32_t* o, int w, int y, int z, int c, int L, int W, uint32_t* centre) {
    const int par = (y + z + c) & 1;
    const int yp = y + 1 == L ? 0 : y + 1, ym = y == 0 ? L - 1 : y - 1;
    const int zp = z + 1 == L ? 0 : z + 1, zm = z == 0 ? L - 1 : z - 1;
    const int row = W * (y + L * z);
    const uint32_t cw = o[row + w];
    uint32_t sh;
    if (par == 0) sh = __funnelshift_r(o[row + (w == 0 ? W - 1 : w - 1)], cw, 24);      // site xh-1
    else sh = __funnelshift_r(cw, o[row + (w + 1 == W ? 0 : w + 1)], 8);                // site xh+1
    *centre = cw;
    return cw + sh + o[W * (yp + L * z) + w] + o[W * (ym + L * z) + w] + o[W * (y + L * zp) + w] + o[W * (y + L * zm) + w];
}

template <int KIND, bool MULTI = false>
__global__ void __launch_bounds__(kSmallMaxThreads, 1) k_sweep_small(const View v, const SmallParams sp) {
    extern __shared__ __align__(16) uint8_t sm_raw[];
    const int tid = threadIdx.x, T = blockDim.x;
    const int L = v.L, W = v.W, NW = (int)(v.Nh >> 2);
    uint32_t* s_spin = reinterpret_cast<uint32_t*>(sm_raw);                    // [2][NW] words of 0/1 bytes
    uint32_t* s_tab = s_spin + 2 * NW;                                         // bimodal: etab[32]; Gaussian: GaussEntry[16]
    long long* s_red = reinterpret_cast<long long*>(s_tab + 64);               // [3][32] warp partial sums
    __shared__ int s_last;

    // which replica: by rank, or (replica shard) by stored slot -- as in sweep_res.cuh
    const int d = blockIdx.x / v.n_it, q0 = blockIdx.x % v.n_it;
    int slot, tr;
    if (v.shard) { slot = v.stored_slot(q0); tr = d * v.R + v.r2t[d * v.R + slot]; }
    else { tr = d * v.R + q0; slot = v.t2r[tr]; }
    const long long ds = (long long)d * v.Rs + v.stored_index(slot);
    const uint32_t k0 = v.keys[2 * d], k1 = v.keys[2 * d + 1];
    const long long fbase0 = (long long)d * 2 * v.Nh;

    // ---- load: global (0/1 bytes; the bit-packed layout is read by the plane-run kernel only) -> shared ----------
    {
        const uint32_t* src = reinterpret_cast<const uint32_t*>(v.spins + ds * 2 * v.Nh);
        for (int i = tid; i < 2 * NW; i += T) s_spin[i] = __ldcg(src + i);
    }
    if (KIND == 0) { if (tid < 32) s_tab[tid] = v.etab[(long long)tr * 32 + tid]; }
    else if (tid < 32) s_tab[tid] = reinterpret_cast<const uint32_t*>(v.gtab + (long long)tr * 16)[tid];
    uint32_t never = KIND == 0 ? v.never[tr] : 0u;
    float band = KIND == 0 ? 0.f : v.band[tr];
    double beta = v.beta[tr];
    __syncthreads();

    const int nseg = MULTI ? sp.nseg : 1;            // several moves per launch: the MULTI instantiation, cooperative launches only
    for (int seg = 0; seg < nseg; ++seg) {
    const int p_begin = !MULTI || seg == 0 ? 0 : sp.first2 + (seg - 1) * sp.period2;
    const int p_end = !MULTI ? sp.phases : sp.first2 + seg * sp.period2;
    // ---- the phases ------------------------------------------------------------------------------------
    for (int p = p_begin; p < p_end; ++p) {
        const int c = p & 1;
        const uint32_t sweep = sp.sweep0 + (uint32_t)(p >> 1);
        uint32_t* mine = s_spin + c * NW;
        const uint32_t* other = s_spin + (1 - c) * NW;
        const long long fbase = fbase0 + (long long)c * v.Nh;
        for (int q = tid; q < NW; q += T) {
            const int w = q % W, y = (q / W) % L, z = q / (W * L);
            uint32_t centre;
            const uint32_t sum = small_neighbours(other, w, y, z, c, L, W, &centre);
            const uint32_t s4 = mine[q];
            const Words4 r = philox4x32_10(k0, k1, (uint32_t)q, sweep, (uint32_t)slot, c == 0 ? kDomColour0 : kDomColour1);
            uint32_t flips = 0;
            if (KIND == 0) {
                const uint32_t f4 = *reinterpret_cast<const uint32_t*>(v.fieldb + fbase + 4 * q);
                const uint32_t idx4 = sum + (s4 << 3) + f4;
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (bimodal_accept(s_tab, never, (int)byte_of(idx4, k), pick_word(r, k))) flips |= 1u << (8 * k);
            } else {
                const GaussEntry* gt = reinterpret_cast<const GaussEntry*>(s_tab);
                const float4 fa = *reinterpret_cast<const float4*>(v.fielda + fbase + 4 * q);
                const float a4[4] = {fa.x, fa.y, fa.z, fa.w};
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (gauss_accept(v, gt, band, beta, (int)byte_of(s4, k), (int)byte_of(sum, k), a4[k], v.fieldg[fbase + 4 * q + k], pick_word(r, k)))
                        flips |= 1u << (8 * k);
            }
            mine[q] = s4 ^ flips;
        }
        __syncthreads();
    }

    if (!MULTI || seg == nseg - 1) {
    // ---- store back ----------------------------------------------------------------------------------------
        {
            uint32_t* dst = reinterpret_cast<uint32_t*>(v.spins + ds * 2 * v.Nh);
            for (int i = tid; i < 2 * NW; i += T) dst[i] = s_spin[i];
        }

    }

    // ---- measurement (S5): every bond has exactly one colour-0 end -----------------------------------------
    if (sp.measure) {
        const uint32_t* c0 = s_spin;
        const uint32_t* c1 = s_spin + NW;
        long long eb = 0, ef = 0, ms = 0;
        for (int q = tid; q < NW; q += T) {
            const int w = q % W, y = (q / W) % L, z = q / (W * L);
            uint32_t c;
            const uint32_t sum = small_neighbours(c1, w, y, z, 0, L, W, &c);
            const uint32_t s0 = c0[q];
            const int sn = dot4(s0, sum), ss = dot4(s0, 0x01010101u), nn = dot4(sum, 0x01010101u), s1s = dot4(c, 0x01010101u);
            eb += 4 * sn - 12 * ss - 2 * nn + 24;            // sum over the word of (2 s - 1)(2 n1 - 6)
            ms += 2 * (ss + s1s) - 8;
            if (KIND == 0) {
                const uint32_t h0 = *reinterpret_cast<const uint32_t*>(v.fieldb + fbase0 + 4 * q) >> 4;
                const uint32_t h1 = *reinterpret_cast<const uint32_t*>(v.fieldb + fbase0 + v.Nh + 4 * q) >> 4;
                ef += 4 * dot4(h0, s0) - 2 * dot4(h0, 0x01010101u) - 2 * ss + 4;      // sum (2h-1)(2s-1) per site
                ef += 4 * dot4(h1, c) - 2 * dot4(h1, 0x01010101u) - 2 * s1s + 4;
            } else {
                const int4 g0 = *reinterpret_cast<const int4*>(v.fieldg + fbase0 + 4 * q);
                const int4 g1 = *reinterpret_cast<const int4*>(v.fieldg + fbase0 + v.Nh + 4 * q);
                const int gg0[4] = {g0.x, g0.y, g0.z, g0.w}, gg1[4] = {g1.x, g1.y, g1.z, g1.w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    ef += ((s0 >> (8 * k)) & 1u) ? (long long)gg0[k] : -(long long)gg0[k];
                    ef += ((c >> (8 * k)) & 1u) ? (long long)gg1[k] : -(long long)gg1[k];
                }
            }
        }
        eb = warp_sum(eb); ef = warp_sum(ef); ms = warp_sum(ms);
        if ((tid & 31) == 0) { s_red[tid >> 5] = eb; s_red[32 + (tid >> 5)] = ef; s_red[64 + (tid >> 5)] = ms; }
        __syncthreads();
        if (tid < 3) {
            long long t = 0;
            for (int i = 0; i < (T + 31) / 32; ++i) t += s_red[32 * tid + i];
            atomicAdd(reinterpret_cast<unsigned long long*>(v.acc + ((long long)d * v.R + slot) * 3 + tid), (unsigned long long)t);
        }
    }

    if (!MULTI || seg == nseg - 1) break;
    // ---- an exchange step inside the launch: every CTA's sums are in View::acc once all have arrived; the last one runs the
    // step and releases the flag word; then this replica's new rank, table, guard band and beta (the lattice keeps its slot)
    {
        __threadfence();
        __syncthreads();
        if (tid == 0) s_last = (atomicAdd(sp.ticket, 1u) == gridDim.x * (unsigned)(seg + 1) - 1u) ? 1 : 0;
        __syncthreads();
        const uint32_t xwant = (sp.epoch << 8) | (uint32_t)(seg + 1);
        if (s_last) {
            __threadfence();
            for (int dd = 0; dd < v.D; ++dd) {
                exchange_member(v, dd, sp.xstep + (uint32_t)seg, sp.xrow + seg, 1);
                __syncthreads();
            }
            __threadfence();
            if (tid == 0) st_release_gpu(sp.xflag, xwant);
        } else if (tid == 0) {
            int polls = 0;
            while (ld_acquire_gpu(sp.xflag) != xwant) {
                backoff();
                if (++polls > (1 << 22)) { atomicOr(sp.diag, 1ull); break; }
            }
        }
        __syncthreads();
        tr = d * v.R + __ldcg(v.r2t + d * v.R + slot);
        if (KIND == 0) { if (tid < 32) s_tab[tid] = v.etab[(long long)tr * 32 + tid]; }
        else if (tid < 32) s_tab[tid] = reinterpret_cast<const uint32_t*>(v.gtab + (long long)tr * 16)[tid];
        never = KIND == 0 ? v.never[tr] : 0u;
        band = KIND == 0 ? 0.f : v.band[tr];
        beta = v.beta[tr];
        __syncthreads();
    }
    }

    // ---- exchange step by the CTA that arrives last -------------------------------------------------------------
    if (sp.exchange) {
        __threadfence();
        __syncthreads();
        if (tid == 0) s_last = (atomicAdd(sp.ticket, 1u) == gridDim.x * (unsigned)nseg - 1u) ? 1 : 0;
        __syncthreads();
        if (s_last) {
            __threadfence();
            for (int dd = 0; dd < v.D; ++dd) {
                exchange_member(v, dd, sp.xstep + (uint32_t)(nseg - 1), sp.xrow + (nseg - 1), 1);
                __syncthreads();
            }
            if (tid == 0) *sp.ticket = 0u;
        }
    }
}

}  // namespace rfim
