// kernels_ref.cuh -- the straightforward device kernels: one thread per site (any even L) and one
// thread per 4-site word (L % 8 == 0), one launch per colour.  They are the in-library reference
// the tuned kernels (sweep_res.cuh, sweep_small.cuh, sweep_flow.cuh) are checked against, and they serve every lattice size the
// tuned kernels do not.  All decisions follow DESIGN.md S2-S6.
#pragma once
#include <cstdint>
#include "philox.cuh"
#include "view.h"

namespace rfim {

// ---- small helpers -------------------------------------------------------------------------

__device__ __forceinline__ float ex2_approx(float x) {
#if defined(__CUDA_ARCH__)
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
#else
    return exp2f(x);
#endif
}

// exact rule of DESIGN.md S3 for one Gaussian-field attempt, every operation separately rounded
__device__ __noinline__ bool gauss_accept_exact(const View& v, int sbit, int n1, int32_t g, double beta, uint32_t u) {
    const double s = sbit ? 1.0 : -1.0;
    const double nsum = (double)(2 * n1 - 6);
    const double local = __dadd_rn(__dmul_rn(v.J, nsum), __dmul_rn(v.hs, (double)g));
    const double dE = __dmul_rn(__dmul_rn(2.0, s), local);
    const double x = __dmul_rn(dE, beta);
    const double p = exp(-x);
    atomicAdd(&v.diag[1], 1ull);
    if (p >= 1.0) return true;
    const double P = p * 4294967296.0;
    if (fabs(P - ((double)u + 1.0)) < 1e-5) atomicAdd(&v.diag[2], 1ull);
    return (double)u < floor(P);
}

// Gaussian attempt: float estimate with a rigorous guard band, exact binary64 rule inside the band.
// tab = this rank's 16-entry table, a = (float)g (exact; the table's y carries hs).
__device__ __forceinline__ bool gauss_accept(const View& v, const GaussEntry* __restrict__ tab, float band, double beta,
                                             int sbit, int n1, float a, int32_t g, uint32_t u) {
    const GaussEntry e = tab[n1 | (sbit << 3)];
    const float arg = fmaf(a, e.y, e.x);
    const float P = ex2_approx(arg);
    const float d = __uint2float_rn(u) - P;
    if (fabsf(d) < band) return gauss_accept_exact(v, sbit, n1, g, beta, u);
    return d < 0.0f;
}

__device__ __forceinline__ bool bimodal_accept(const uint32_t* __restrict__ etab, uint32_t never, int idx, uint32_t u) {
    return (u <= etab[idx]) && !((never >> idx) & 1u);
}

// ---- generic sweep: one thread per same-colour site, any even L --------------------------------
// grid.y enumerates (member d, rank t); grid-stride over j in [0, Nh).
__global__ void k_sweep_site(View v, int colour, uint32_t sweep) {
    const int d = blockIdx.y / v.n, t = blockIdx.y % v.n;
    const int slot = v.t2r[d * v.R + t];
    const long long Nh = v.Nh;
    uint8_t* mine = v.spins + ((long long)(d * v.R + slot) * 2 + colour) * Nh;
    const uint8_t* other = v.spins + ((long long)(d * v.R + slot) * 2 + (1 - colour)) * Nh;
    const long long fbase = ((long long)d * 2 + colour) * Nh;
    const int tr = d * v.R + t;
    const uint32_t k0 = v.keys[2 * d], k1 = v.keys[2 * d + 1];
    const int L = v.L, Lh = v.Lh;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < Nh; j += (long long)gridDim.x * blockDim.x) {
        const int xh = (int)(j % Lh);
        const int y = (int)((j / Lh) % L);
        const int z = (int)(j / ((long long)Lh * L));
        const int par = (y + z + colour) & 1;
        int xo = xh - 1 + 2 * par;
        xo = xo < 0 ? xo + Lh : (xo >= Lh ? xo - Lh : xo);
        const int yp = y + 1 == L ? 0 : y + 1, ym = y == 0 ? L - 1 : y - 1;
        const int zp = z + 1 == L ? 0 : z + 1, zm = z == 0 ? L - 1 : z - 1;
        const long long row = (long long)Lh * (y + (long long)L * z);
        const int n1 = other[row + xh] + other[row + xo]
                     + other[(long long)Lh * (yp + (long long)L * z) + xh] + other[(long long)Lh * (ym + (long long)L * z) + xh]
                     + other[(long long)Lh * (y + (long long)L * zp) + xh] + other[(long long)Lh * (y + (long long)L * zm) + xh];
        const int sbit = mine[j];
        const Words4 w = philox4x32_10(k0, k1, (uint32_t)(j >> 2), sweep, (uint32_t)slot,
                                       colour == 0 ? kDomColour0 : kDomColour1);
        const uint32_t u = pick_word(w, (uint32_t)(j & 3));
        bool acc;
        if (v.kind == 0) {
            const int idx = n1 | (sbit << 3) | v.fieldb[fbase + j];
            acc = bimodal_accept(v.etab + (long long)tr * 32, v.never[tr], idx, u);
        } else {
            acc = gauss_accept(v, v.gtab + (long long)tr * 16, v.band[tr], v.beta[tr], sbit, n1,
                               v.fielda[fbase + j], v.fieldg[fbase + j], u);
        }
        if (acc) mine[j] = (uint8_t)(sbit ^ 1);
    }
}

// ---- word sweep: one thread per 32-bit word = 4 same-colour sites = one Philox call (L % 8 == 0) --
__device__ __forceinline__ uint32_t byte_of(uint32_t w, int k) { return (w >> (8 * k)) & 0xFFu; }

__global__ void k_sweep_word(View v, int colour, uint32_t sweep) {
    const int d = blockIdx.y / v.n, t = blockIdx.y % v.n;
    const int slot = v.t2r[d * v.R + t];
    const long long NW = v.Nh >> 2;
    uint32_t* mine = reinterpret_cast<uint32_t*>(v.spins + ((long long)(d * v.R + slot) * 2 + colour) * v.Nh);
    const uint32_t* other = reinterpret_cast<const uint32_t*>(v.spins + ((long long)(d * v.R + slot) * 2 + (1 - colour)) * v.Nh);
    const long long fbase = ((long long)d * 2 + colour) * v.Nh;
    const int tr = d * v.R + t;
    const uint32_t k0 = v.keys[2 * d], k1 = v.keys[2 * d + 1];
    const int L = v.L, W = v.W;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < NW; q += (long long)gridDim.x * blockDim.x) {
        const int w = (int)(q % W);
        const int y = (int)((q / W) % L);
        const int z = (int)(q / ((long long)W * L));
        const int par = (y + z + colour) & 1;
        const int yp = y + 1 == L ? 0 : y + 1, ym = y == 0 ? L - 1 : y - 1;
        const int zp = z + 1 == L ? 0 : z + 1, zm = z == 0 ? L - 1 : z - 1;
        const long long row = (long long)W * (y + (long long)L * z);
        const uint32_t c = other[row + w];
        // the x-neighbour on the far side: parity 0 -> bytes shifted up by one (xh-1), parity 1 -> down (xh+1)
        uint32_t sh;
        if (par == 0) {
            const uint32_t p = other[row + (w == 0 ? W - 1 : w - 1)];
            sh = (c << 8) | (p >> 24);
        } else {
            const uint32_t nx = other[row + (w + 1 == W ? 0 : w + 1)];
            sh = (c >> 8) | (nx << 24);
        }
        const uint32_t sum = c + sh
                           + other[(long long)W * (yp + (long long)L * z) + w] + other[(long long)W * (ym + (long long)L * z) + w]
                           + other[(long long)W * (y + (long long)L * zp) + w] + other[(long long)W * (y + (long long)L * zm) + w];
        const uint32_t s4 = mine[q];
        const Words4 r = philox4x32_10(k0, k1, (uint32_t)q, sweep, (uint32_t)slot, colour == 0 ? kDomColour0 : kDomColour1);
        uint32_t flips = 0;
        if (v.kind == 0) {
            const uint32_t f4 = *reinterpret_cast<const uint32_t*>(v.fieldb + fbase + 4 * q);
            const uint32_t idx4 = sum + (s4 << 3) + f4;
            const uint32_t* et = v.etab + (long long)tr * 32;
            const uint32_t nv = v.never[tr];
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (bimodal_accept(et, nv, (int)byte_of(idx4, k), pick_word(r, k))) flips |= 1u << (8 * k);
        } else {
            const GaussEntry* gt = v.gtab + (long long)tr * 16;
            const float band = v.band[tr];
            const double beta = v.beta[tr];
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (gauss_accept(v, gt, band, beta, (int)byte_of(s4, k), (int)byte_of(sum, k), v.fielda[fbase + 4 * q + k],
                                 v.fieldg[fbase + 4 * q + k], pick_word(r, k)))
                    flips |= 1u << (8 * k);
        }
        mine[q] = s4 ^ flips;
    }
}

// ---- initial spins (S2, domain 3): one thread per site in natural order ---------------
__global__ void k_init_spins(View v) {
    const int d = blockIdx.y / v.Rs, slot = v.stored_slot(blockIdx.y % v.Rs);   // grid.y = D * (stored slots per member)
    const uint32_t k0 = v.keys[2 * d], k1 = v.keys[2 * d + 1];
    const int L = v.L, Lh = v.Lh;
    uint8_t* base = v.spins + (long long)blockIdx.y * 2 * v.Nh;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < v.N; i += (long long)gridDim.x * blockDim.x) {
        const Words4 w = philox4x32_10(k0, k1, (uint32_t)(i >> 2), 0u, (uint32_t)slot, kDomInitSpins);
        const uint32_t bit = pick_word(w, (uint32_t)(i & 3)) >> 31;
        const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long long)L * L));
        const int c = (x + y + z) & 1;
        base[(long long)c * v.Nh + (x >> 1) + (long long)Lh * (y + (long long)L * z)] = (uint8_t)bit;
    }
}

// ---- natural-order +-1 int8  <->  colour-separated 0/1 bytes (or bits), slots [first, first+count) --------
__global__ void k_export_spins(View v, int first, int8_t* __restrict__ out) {
    const int ds = first + blockIdx.y;     // linear d*R + slot
    const int L = v.L, Lh = v.Lh;
    const long long b0 = (long long)ds * 2 * v.Nh;
    int8_t* o = out + (long long)blockIdx.y * v.N;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < v.N; i += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long long)L * L));
        const int c = (x + y + z) & 1;
        const long long j = b0 + (long long)c * v.Nh + (x >> 1) + (long long)Lh * (y + (long long)L * z);
        const int up = v.packed ? (v.spins[j >> 3] >> (j & 7)) & 1 : v.spins[j];
        o[i] = up ? 1 : -1;
    }
}

__global__ void k_import_spins(View v, int first, const int8_t* __restrict__ in) {
    const int ds = first + blockIdx.y;
    const int L = v.L, Lh = v.Lh;
    const int8_t* src = in + (long long)blockIdx.y * v.N;
    if (v.packed) {                        // one thread per packed byte: eight same-colour sites
        uint8_t* base = v.spins + (long long)ds * (v.N >> 3);
        for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < (v.N >> 3); b += (long long)gridDim.x * blockDim.x) {
            const int c = (int)(b / (v.Nh >> 3));
            const long long j0 = (b % (v.Nh >> 3)) * 8;
            uint32_t bits = 0;
            for (int t = 0; t < 8; ++t) {
                const long long j = j0 + t;
                const int xh = (int)(j % Lh), y = (int)((j / Lh) % L), z = (int)(j / ((long long)Lh * L));
                const int x = 2 * xh + ((y + z + c) & 1);
                if (src[x + (long long)L * (y + (long long)L * z)] > 0) bits |= 1u << t;
            }
            base[b] = (uint8_t)bits;
        }
        return;
    }
    uint8_t* base = v.spins + (long long)ds * 2 * v.Nh;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < v.N; i += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long long)L * L));
        const int c = (x + y + z) & 1;
        base[(long long)c * v.Nh + (x >> 1) + (long long)Lh * (y + (long long)L * z)] = src[i] > 0 ? 1 : 0;
    }
}

// ---- the same with the HOST side bit-packed: bit (i & 7) of byte (i >> 3) of a lattice = 1 iff s_i = +1, i the natural
// site index x + L (y + L z): an eighth of the PCIe traffic of the int8 interface.  N is a multiple of 8 (L is even).
__global__ void k_export_bits(View v, int first, uint8_t* __restrict__ out) {
    const int ds = first + blockIdx.y;
    const int L = v.L, Lh = v.Lh;
    const long long b0 = (long long)ds * 2 * v.Nh;
    uint8_t* o = out + (long long)blockIdx.y * (v.N >> 3);
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < (v.N >> 3); b += (long long)gridDim.x * blockDim.x) {
        uint32_t bits = 0;
        for (int t = 0; t < 8; ++t) {
            const long long i = 8 * b + t;
            const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long long)L * L));
            const int c = (x + y + z) & 1;
            const long long j = b0 + (long long)c * v.Nh + (x >> 1) + (long long)Lh * (y + (long long)L * z);
            const uint32_t up = v.packed ? (v.spins[j >> 3] >> (j & 7)) & 1u : v.spins[j];
            bits |= up << t;
        }
        o[b] = (uint8_t)bits;
    }
}

__global__ void k_import_bits(View v, int first, const uint8_t* __restrict__ in) {
    const int ds = first + blockIdx.y;
    const int L = v.L, Lh = v.Lh;
    const uint8_t* src = in + (long long)blockIdx.y * (v.N >> 3);
    // one thread per group of eight same-colour sites j0 .. j0+7 (one packed byte, or eight bytes of the byte layout)
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < (v.N >> 3); b += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(b / (v.Nh >> 3));
        const long long j0 = (b % (v.Nh >> 3)) * 8;
        uint32_t bits = 0;
        for (int t = 0; t < 8; ++t) {
            const long long j = j0 + t;
            const int xh = (int)(j % Lh), y = (int)((j / Lh) % L), z = (int)(j / ((long long)Lh * L));
            const long long i = 2 * xh + ((y + z + c) & 1) + (long long)L * (y + (long long)L * z);
            bits |= ((src[i >> 3] >> (i & 7)) & 1u) << t;
        }
        if (v.packed) {
            v.spins[(long long)ds * (v.N >> 3) + b] = (uint8_t)bits;
        } else {
            uint8_t* dst = v.spins + (long long)ds * 2 * v.Nh + (long long)c * v.Nh + j0;
            for (int t = 0; t < 8; ++t) dst[t] = (uint8_t)((bits >> t) & 1u);
        }
    }
}

// ---- the same two conversions for L % 16 == 0 (L = 16, 32, 64: the sizes the host interface is timed on): one thread per 16
// consecutive sites of a row of the natural order = two bytes of the bit format = eight sites of each colour (one aligned
// 8-byte group of the byte layout, or one byte of the packed layout).  Even x belong to colour (y+z)&1, odd x to the other.
__device__ __forceinline__ uint32_t bits_spread8(uint32_t v) {          // bit m of v -> bit 2m
    v = (v | (v << 4)) & 0x0F0Fu; v = (v | (v << 2)) & 0x3333u; v = (v | (v << 1)) & 0x5555u;
    return v;
}
__device__ __forceinline__ uint32_t bits_compact8(uint32_t v) {         // bit 2m of v -> bit m
    v &= 0x5555u; v = (v | (v >> 1)) & 0x3333u; v = (v | (v >> 2)) & 0x0F0Fu; v = (v | (v >> 4)) & 0x00FFu;
    return v;
}
__device__ __forceinline__ uint32_t bytes01_to_bits8(uint2 w) {        // eight bytes of 0/1 -> eight bits
    return ((((w.x & 0x01010101u) * 0x01020408u) >> 24) & 0xFu) | (((((w.y & 0x01010101u) * 0x01020408u) >> 24) & 0xFu) << 4);
}
__device__ __forceinline__ uint2 bits8_to_bytes01(uint32_t b) {
    return make_uint2(((b & 0xFu) * 0x00204081u) & 0x01010101u, (((b >> 4) & 0xFu) * 0x00204081u) & 0x01010101u);
}
__global__ void k_export_bits16(View v, int first, uint8_t* __restrict__ out) {
    const int ds = first + blockIdx.y;
    const int L = v.L, Lh = v.Lh, cpr = L >> 4;                          // 16-site chunks per row
    const long long chunks = v.N >> 4;
    unsigned short* o = reinterpret_cast<unsigned short*>(out + (long long)blockIdx.y * (v.N >> 3));
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < chunks; q += (long long)gridDim.x * blockDim.x) {
        const long long row = q / cpr;                                   // y + L z
        const int xq = (int)(q - row * cpr), y = (int)(row % L), z = (int)(row / L);
        const int ce = (y + z) & 1;                                      // colour of the even x of this row
        const long long j0 = (long long)Lh * row + 8 * xq;               // same-colour index of the chunk's first site, both colours
        uint32_t be, bo;
        if (v.packed) {
            const uint8_t* base = v.spins + (long long)ds * (v.N >> 3);
            be = base[((long long)ce * v.Nh + j0) >> 3];
            bo = base[((long long)(1 - ce) * v.Nh + j0) >> 3];
        } else {
            const uint8_t* base = v.spins + (long long)ds * 2 * v.Nh;
            be = bytes01_to_bits8(*reinterpret_cast<const uint2*>(base + (long long)ce * v.Nh + j0));
            bo = bytes01_to_bits8(*reinterpret_cast<const uint2*>(base + (long long)(1 - ce) * v.Nh + j0));
        }
        o[q] = (unsigned short)(bits_spread8(be) | (bits_spread8(bo) << 1));
    }
}
__global__ void k_import_bits16(View v, int first, const uint8_t* __restrict__ in) {
    const int ds = first + blockIdx.y;
    const int L = v.L, Lh = v.Lh, cpr = L >> 4;
    const long long chunks = v.N >> 4;
    const unsigned short* src = reinterpret_cast<const unsigned short*>(in + (long long)blockIdx.y * (v.N >> 3));
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < chunks; q += (long long)gridDim.x * blockDim.x) {
        const long long row = q / cpr;
        const int xq = (int)(q - row * cpr), y = (int)(row % L), z = (int)(row / L);
        const int ce = (y + z) & 1;
        const long long j0 = (long long)Lh * row + 8 * xq;
        const uint32_t w = src[q];
        const uint32_t be = bits_compact8(w), bo = bits_compact8(w >> 1);
        if (v.packed) {
            uint8_t* base = v.spins + (long long)ds * (v.N >> 3);
            base[((long long)ce * v.Nh + j0) >> 3] = (uint8_t)be;
            base[((long long)(1 - ce) * v.Nh + j0) >> 3] = (uint8_t)bo;
        } else {
            uint8_t* base = v.spins + (long long)ds * 2 * v.Nh;
            *reinterpret_cast<uint2*>(base + (long long)ce * v.Nh + j0) = bits8_to_bytes01(be);
            *reinterpret_cast<uint2*>(base + (long long)(1 - ce) * v.Nh + j0) = bits8_to_bytes01(bo);
        }
    }
}

// natural-order +-1 int8 <-> device layout, L % 16 == 0: one thread per 16 consecutive sites of a row (one 16-byte load or store)
__device__ __forceinline__ uint32_t bytes01_to_pm1(uint32_t w) { return ((w ^ 0x01010101u) * 0xFFu) | 0x01010101u; }   // 1 -> 0x01, 0 -> 0xFF
__device__ __forceinline__ uint32_t pm1_to_bytes01(uint32_t w) {                                                       // s > 0 -> 1, s <= 0 -> 0, per byte
    return ((((w & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) & ~w & 0x80808080u) >> 7);
}
__global__ void k_export_spins16(View v, int first, int8_t* __restrict__ out) {
    const int ds = first + blockIdx.y;
    const int L = v.L, Lh = v.Lh, cpr = L >> 4;
    const long long chunks = v.N >> 4;
    uint4* o = reinterpret_cast<uint4*>(out + (long long)blockIdx.y * v.N);
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < chunks; q += (long long)gridDim.x * blockDim.x) {
        const long long row = q / cpr;
        const int xq = (int)(q - row * cpr), y = (int)(row % L), z = (int)(row / L);
        const int ce = (y + z) & 1;
        const long long j0 = (long long)Lh * row + 8 * xq;
        uint2 e, od;
        if (v.packed) {
            const uint8_t* base = v.spins + (long long)ds * (v.N >> 3);
            e = bits8_to_bytes01(base[((long long)ce * v.Nh + j0) >> 3]);
            od = bits8_to_bytes01(base[((long long)(1 - ce) * v.Nh + j0) >> 3]);
        } else {
            const uint8_t* base = v.spins + (long long)ds * 2 * v.Nh;
            e = *reinterpret_cast<const uint2*>(base + (long long)ce * v.Nh + j0);
            od = *reinterpret_cast<const uint2*>(base + (long long)(1 - ce) * v.Nh + j0);
        }
        uint4 n;
        n.x = bytes01_to_pm1(__byte_perm(e.x, od.x, 0x5140)); n.y = bytes01_to_pm1(__byte_perm(e.x, od.x, 0x7362));
        n.z = bytes01_to_pm1(__byte_perm(e.y, od.y, 0x5140)); n.w = bytes01_to_pm1(__byte_perm(e.y, od.y, 0x7362));
        o[q] = n;
    }
}
__global__ void k_import_spins16(View v, int first, const int8_t* __restrict__ in) {
    const int ds = first + blockIdx.y;
    const int L = v.L, Lh = v.Lh, cpr = L >> 4;
    const long long chunks = v.N >> 4;
    const uint4* src = reinterpret_cast<const uint4*>(in + (long long)blockIdx.y * v.N);
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < chunks; q += (long long)gridDim.x * blockDim.x) {
        const long long row = q / cpr;
        const int xq = (int)(q - row * cpr), y = (int)(row % L), z = (int)(row / L);
        const int ce = (y + z) & 1;
        const long long j0 = (long long)Lh * row + 8 * xq;
        uint4 n = src[q];
        n.x = pm1_to_bytes01(n.x); n.y = pm1_to_bytes01(n.y); n.z = pm1_to_bytes01(n.z); n.w = pm1_to_bytes01(n.w);
        const uint2 e = make_uint2(__byte_perm(n.x, n.y, 0x6420), __byte_perm(n.z, n.w, 0x6420));
        const uint2 od = make_uint2(__byte_perm(n.x, n.y, 0x7531), __byte_perm(n.z, n.w, 0x7531));
        if (v.packed) {
            uint8_t* base = v.spins + (long long)ds * (v.N >> 3);
            base[((long long)ce * v.Nh + j0) >> 3] = (uint8_t)bytes01_to_bits8(e);
            base[((long long)(1 - ce) * v.Nh + j0) >> 3] = (uint8_t)bytes01_to_bits8(od);
        } else {
            uint8_t* base = v.spins + (long long)ds * 2 * v.Nh;
            *reinterpret_cast<uint2*>(base + (long long)ce * v.Nh + j0) = e;
            *reinterpret_cast<uint2*>(base + (long long)(1 - ce) * v.Nh + j0) = od;
        }
    }
}

// ---- whole-buffer conversion between the byte and the bit layout (same index j, eight spins per byte) ----------
__global__ void k_pack_bits(const uint8_t* __restrict__ bytes, uint8_t* __restrict__ bits, long long nbits_bytes) {
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < nbits_bytes; b += (long long)gridDim.x * blockDim.x) {
        const uint2 w = *reinterpret_cast<const uint2*>(bytes + 8 * b);
        const uint32_t lo = ((w.x & 0x01010101u) * 0x01020408u) >> 24, hi = ((w.y & 0x01010101u) * 0x01020408u) >> 24;
        bits[b] = (uint8_t)((lo & 0xFu) | ((hi & 0xFu) << 4));
    }
}
__global__ void k_unpack_bits(const uint8_t* __restrict__ bits, uint8_t* __restrict__ bytes, long long nbits_bytes) {
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < nbits_bytes; b += (long long)gridDim.x * blockDim.x) {
        const uint32_t q = bits[b];
        uint2 w;
        w.x = ((q & 0xFu) * 0x00204081u) & 0x01010101u;
        w.y = ((q >> 4) * 0x00204081u) & 0x01010101u;
        *reinterpret_cast<uint2*>(bytes + 8 * b) = w;
    }
}

// ---- energy / magnetisation reduction (S5) -----------------------------
// Every directed bond has exactly one colour-0 end, so Eb = sum over colour-0 sites of s_i * (six-neighbour sum).
__device__ __forceinline__ long long warp_sum(long long x) {
#if defined(__CUDA_ARCH__)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xFFFFFFFFu, x, o);
#endif
    return x;
}

__global__ void k_reduce_site(View v) {
    const int d = blockIdx.y / v.n, t = blockIdx.y % v.n;
    const int slot = v.t2r[d * v.R + t];
    if (!v.stores(slot)) return;                                              // a replica shard reduces the slots it stores
    const long long Nh = v.Nh;
    const uint8_t* c0 = v.spins + (long long)(d * v.Rs + v.stored_index(slot)) * 2 * Nh;
    const uint8_t* c1 = c0 + Nh;
    const long long f0 = (long long)d * 2 * Nh, f1 = f0 + Nh;
    const int L = v.L, Lh = v.Lh;
    long long eb = 0, ef = 0, ms = 0;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < Nh; j += (long long)gridDim.x * blockDim.x) {
        const int xh = (int)(j % Lh);
        const int y = (int)((j / Lh) % L);
        const int z = (int)(j / ((long long)Lh * L));
        const int par = (y + z) & 1;
        int xo = xh - 1 + 2 * par;
        xo = xo < 0 ? xo + Lh : (xo >= Lh ? xo - Lh : xo);
        const int yp = y + 1 == L ? 0 : y + 1, ym = y == 0 ? L - 1 : y - 1;
        const int zp = z + 1 == L ? 0 : z + 1, zm = z == 0 ? L - 1 : z - 1;
        const long long row = (long long)Lh * (y + (long long)L * z);
        const int n1 = c1[row + xh] + c1[row + xo]
                     + c1[(long long)Lh * (yp + (long long)L * z) + xh] + c1[(long long)Lh * (ym + (long long)L * z) + xh]
                     + c1[(long long)Lh * (y + (long long)L * zp) + xh] + c1[(long long)Lh * (y + (long long)L * zm) + xh];
        const int s0 = 2 * (int)c0[j] - 1, s1 = 2 * (int)c1[j] - 1;
        eb += s0 * (2 * n1 - 6);
        ms += s0 + s1;
        if (v.kind == 0) {
            ef += (v.fieldb[f0 + j] ? s0 : -s0) + (v.fieldb[f1 + j] ? s1 : -s1);
        } else {
            ef += (long long)s0 * v.fieldg[f0 + j] + (long long)s1 * v.fieldg[f1 + j];
        }
    }
    eb = warp_sum(eb); ef = warp_sum(ef); ms = warp_sum(ms);
    if ((threadIdx.x & 31) == 0) {
        long long* a = v.acc + (long long)(d * v.R + slot) * 3;
        atomicAdd(reinterpret_cast<unsigned long long*>(a + 0), (unsigned long long)eb);
        atomicAdd(reinterpret_cast<unsigned long long*>(a + 1), (unsigned long long)ef);
        atomicAdd(reinterpret_cast<unsigned long long*>(a + 2), (unsigned long long)ms);
    }
}

// ---- exchange step (S6): one CTA per member ------------------
// record != 0: append the row to the time series at index `row`.  The accumulators are consumed (zeroed).
__device__ __forceinline__ void exchange_member(const View& v, int d, uint32_t xstep, long long row, int record) {
    const int n = v.n, R = v.R;
    int32_t* t2r = v.t2r + d * R;
    int32_t* r2t = v.r2t + d * R;
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
        long long* a = v.acc + (long long)(d * R + t2r[t]) * 3;
        const long long eb = __ldcg(a + 0), ef = __ldcg(a + 1), ms = __ldcg(a + 2);   // written by other CTAs' atomics: read at L2
        a[0] = 0; a[1] = 0; a[2] = 0;
        long long* keep = v.last + (long long)(d * R + t2r[t]) * 3;
        keep[0] = eb; keep[1] = ef; keep[2] = ms;
        if (record) {
            long long* s = v.series + ((row * v.D + d) * R + t) * 3;
            s[0] = eb; s[1] = ef; s[2] = ms;
        }
        v.ework[d * R + t] = __dsub_rn(__dmul_rn(-v.J, (double)eb), __dmul_rn(v.hs, (double)ef));
    }
    __syncthreads();
    const uint32_t k0 = v.keys[2 * d], k1 = v.keys[2 * d + 1];
    for (int t = (int)(xstep & 1u) + 2 * (int)threadIdx.x; t + 1 <= n - 1; t += 2 * (int)blockDim.x) {
        const double delta = __dmul_rn(__dsub_rn(v.beta[d * R + t + 1], v.beta[d * R + t]),
                                       __dsub_rn(v.ework[d * R + t + 1], v.ework[d * R + t]));
        v.att[d * R + t] += 1ull;
        bool acc;
        if (delta >= 0.0) {
            acc = true;
        } else {
            const Words4 w = philox4x32_10(k0, k1, (uint32_t)t, xstep, 0u, kDomExchange);
            const double P = exp(delta) * 4294967296.0;
            if (fabs(P - ((double)w.w0 + 1.0)) < 1e-5) atomicAdd(&v.diag[2], 1ull);
            atomicAdd(&v.diag[3], 1ull);
            acc = (double)w.w0 < floor(P);
        }
        if (acc) {
            const int a = t2r[t], b = t2r[t + 1];
            t2r[t] = b; t2r[t + 1] = a;
            r2t[b] = t; r2t[a] = t + 1;
            v.accn[d * R + t] += 1ull;
        }
    }
}

__global__ void k_exchange(View v, uint32_t xstep, long long row, int record) {
    exchange_member(v, (int)blockIdx.x, xstep, row, record);
}

// ---- thermal moments of the measurement series (Eq. 11-13 are built from these on the host) ------
// One CTA per (member d, rank t): out[(d*n + t)*5 + 0..4] = <e>, <e^2>, <|m|>, <m^2>, <m^4> over steps [skip, steps), with
// e = E/N per site (E as in DESIGN.md S5) and m = Msum/N.  Each thread sums a strided subset in step order, then a fixed
// shared-memory tree combines the 256 partial sums: deterministic, and within a few ulp of a sequential sum.
__global__ void k_thermal_moments(View v, long long skip, long long steps, double* __restrict__ out) {
    const int d = blockIdx.x / v.n, t = blockIdx.x % v.n;
    __shared__ double part[5][256];
    double a[5] = {0, 0, 0, 0, 0};
    for (long long q = skip + threadIdx.x; q < steps; q += blockDim.x) {
        const long long* s = v.series + ((q * v.D + d) * v.R + t) * 3;
        const double E = __dsub_rn(__dmul_rn(-v.J, (double)s[0]), __dmul_rn(v.hs, (double)s[1]));
        const double e = E / (double)v.N, m = (double)s[2] / (double)v.N;
        a[0] += e; a[1] += e * e; a[2] += fabs(m); a[3] += m * m; a[4] += (m * m) * (m * m);
    }
    for (int j = 0; j < 5; ++j) part[j][threadIdx.x] = a[j];
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w)
            for (int j = 0; j < 5; ++j) part[j][threadIdx.x] += part[j][threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x < 5) out[(long long)blockIdx.x * 5 + threadIdx.x] = part[threadIdx.x][0] / (double)(steps - skip);
}

}  // namespace rfim
