// rfim_pt.cu -- host side of librfimpt.so: the C ABI of include/rfim_pt.h.
// Handle, device buffers, acceptance tables (binary64 on the host, S3), kernel launch
// sequencing for sweep / reduce / exchange, the adaptation rule (S8), getters.
// No part of this file includes, links or calls anything under oracle/.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/rfim_pt.h"
#include "kernels_ref.cuh"
#include "launch.h"
#include "philox.cuh"
#include "sweep_flow.cuh"
#include "sweep_res.cuh"
#include "sweep_small.cuh"
#include "view.h"

using namespace rfim;

namespace {

rfim_pt_alloc_fn g_alloc = nullptr;
rfim_pt_free_fn g_free = nullptr;

constexpr double kTwo32 = 4294967296.0;
constexpr double kFieldScale = 1048576.0;   // 2^20
constexpr int32_t kFieldClamp = 8 * 1048576;
constexpr int kResMaxGrid = 255;            // owners are stored in 8 bits (sweep_res.cuh)
constexpr int kResFusedExchangeMaxD = 4;    // the last CTA runs the exchange step itself for batches up to this size

}  // namespace

struct rfim_pt {
    int L = 0, R = 0, n = 0, D = 1, kind = 0;
    long long N = 0, Nh = 0;
    double J = 0, h = 0;
    std::vector<uint64_t> seeds;
    cudaStream_t stream = nullptr;
    bool have_T = false;
    std::vector<int32_t> field_nat;   // [D][N] natural order: +-1 or g_i
    std::vector<double> amax;         // [D] max |hs * g_i|
    std::vector<double> T;            // [D][R] by rank
    View v{};
    std::vector<void*> owned;         // every device allocation, released in destroy
    int8_t* stage = nullptr;          // device staging for spin import/export
    int slot0 = 0, Rs = 0;            // stored slots (replica shard: slot0 + j * sstride, j < Rs; else 0, R)
    int sstride = 1;                  // 1: contiguous window; G: round-robin deal over G ranks
    int rank = 0, world = 1;          // replica shard: this rank, number of ranks
    bool shard = false;
    rfim_pt_gather_fn gather = nullptr;   // shard: completes View::acc across ranks before an exchange step
    void* gather_user = nullptr;
    rfim_pt_bcast_fn bcast = nullptr;     // shard: hands one lattice from its owner to every rank (inserting adaptation)
    void* bcast_user = nullptr;
    // shard, native route: the library calls NCCL itself (no host callback per exchange step)
    void* nccl_comm = nullptr;
    int (*nccl_all_gather)(const void*, void*, size_t, int, void*, cudaStream_t) = nullptr;
    int (*nccl_broadcast)(const void*, void*, size_t, int, int, void*, cudaStream_t) = nullptr;
    long long* terms_all = nullptr;   // round-robin shard: [world][Rs][3] rank-major copy of the energy terms for the all-gather
    std::vector<double> trial_rates;  // [D][R]: exchange rates of the last adaptation trial (rfim_pt_get_trial_rates)
    int trial_n = 0;
    size_t acc_rows = 0;              // rows of View::acc (>= R; padded to a whole number of shards)
    double* moments_dev = nullptr;    // thermal moments scratch (rfim_pt_thermal_moments)
    uint8_t* unpacked = nullptr;      // packed mode: byte-layout scratch for the stand-alone reduction (allocated on first use)
    size_t stage_bytes = 0;
    uint64_t sweep_g = 0, xstep = 0;
    long long series_steps = 0, series_cap = 0;
    int adapt_k = 10, adapt_a = 4;
    int packing = 8, variant = 0;
    uint64_t launches = 0;
    uint32_t* flow_prog = nullptr;    // [D][R][32] progress words of the flow kernel
    uint32_t flow_epoch = 0;
    int flow_rr = 4;                  // replicas per work item
    bool has_never = false;           // some reachable bimodal table entry has threshold 0
    float* fielda_res = nullptr;      // resident-kernel copies of the field (task order), L = 32 or 64
    uint8_t* fieldb_res = nullptr;
    long long* gsum_res = nullptr;    // Gaussian: [D][L] sum of g_i over plane z (the resident kernel measures Ef = 2 * sum over up spins - this)
    uint32_t* res_prog = nullptr;     // [kResMaxGrid] progress words of the resident kernel
    uint32_t res_epoch = 0;
    bool terms_fresh = false;         // View::last holds the energy terms of the CURRENT lattices (last call ended on an exchange step)
    int res_grid_limit = 0;           // 0 = one CTA per SM
    int res_partition = 0;            // resident kernel: 0 automatic, 1 equal runs of planes, 2 whole replicas per CTA
    int res_multi = 1;                // != 0 allows several parallel-tempering moves per launch (resident and small-lattice kernels)
    int small_per_sm = -1;            // small-lattice kernel: CTAs per SM (occupancy), -1 = not asked yet
    int sm_count = 0, smem_optin = 0;
    std::string err;
};

namespace {

int fail(rfim_pt* h, int code, const std::string& msg) {
    if (h) h->err = msg;
    return code;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(h, RFIM_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));        \
    } while (0)

void* dev_alloc(size_t bytes) {
    if (bytes == 0) bytes = 16;
    if (g_alloc) return g_alloc(bytes);
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) return nullptr;
    return p;
}
void dev_free(void* p) {
    if (!p) return;
    if (g_free) g_free(p); else cudaFree(p);
}

template <class Tp>
int alloc_into(rfim_pt* h, Tp** out, size_t count) {
    void* p = dev_alloc(count * sizeof(Tp));
    if (!p) return fail(h, RFIM_ENOMEM, "device allocation failed");
    h->owned.push_back(p);
    *out = reinterpret_cast<Tp*>(p);
    return RFIM_OK;
}
void release(rfim_pt* h, void* p) {
    auto it = std::find(h->owned.begin(), h->owned.end(), p);
    if (it != h->owned.end()) h->owned.erase(it);
    dev_free(p);
}

inline long long layout_index(const rfim_pt* h, int x, int y, int z, int* colour) {
    *colour = (x + y + z) & 1;
    return (long long)(x >> 1) + (long long)(h->L / 2) * (y + (long long)h->L * z);
}

// position of site (x,y,z) inside one member's field copy in the resident kernel's task order (sweep_res.cuh):
// [colour][z][class s = (y+z)&1][word w = xh/4][row i = y/2][site xh%4], i.e. 16 bytes (bimodal: [piece xh/16][i][xh%16])
inline long long res_field_index(const rfim_pt* h, int x, int y, int z) {
    const int L = h->L, LH = L / 2, c = (x + y + z) & 1, xh = x >> 1, s = (y + z) & 1, i = y >> 1;
    const long long blk = ((long long)c * L + z) * 2 + s;              // block of L/2 rows x L/2 sites
    if (h->kind == RFIM_FIELD_BIMODAL) return ((blk * (L / 32) + xh / 16) * LH + i) * 16 + xh % 16;
    return ((blk * (L / 8) + xh / 4) * LH + i) * 4 + xh % 4;
}

dim3 grid_for(long long work, int ny, int threads = 256) {
    long long bx = (work + threads - 1) / threads;
    if (bx < 1) bx = 1;
    if (bx > 4096) bx = 4096;
    return dim3((unsigned)bx, (unsigned)ny, 1);
}

// natural-order bit format <-> device layout: the 16-site kernels for L % 16 == 0, the generic per-bit ones otherwise
void launch_export_bits(rfim_pt* h, int ny, int first, uint8_t* out) {
    if (h->L % 16 == 0) k_export_bits16<<<grid_for(h->N / 16, ny), 256, 0, h->stream>>>(h->v, first, out);
    else k_export_bits<<<grid_for(h->N / 8, ny), 256, 0, h->stream>>>(h->v, first, out);
}
void launch_import_bits(rfim_pt* h, int ny, int first, const uint8_t* in) {
    if (h->L % 16 == 0) k_import_bits16<<<grid_for(h->N / 16, ny), 256, 0, h->stream>>>(h->v, first, in);
    else k_import_bits<<<grid_for(h->N / 8, ny), 256, 0, h->stream>>>(h->v, first, in);
}

void launch_export_spins(rfim_pt* h, int ny, int first, int8_t* out) {
    if (h->L % 16 == 0) k_export_spins16<<<grid_for(h->N / 16, ny), 256, 0, h->stream>>>(h->v, first, out);
    else k_export_spins<<<grid_for(h->N, ny), 256, 0, h->stream>>>(h->v, first, out);
}
void launch_import_spins(rfim_pt* h, int ny, int first, const int8_t* in) {
    if (h->L % 16 == 0) k_import_spins16<<<grid_for(h->N / 16, ny), 256, 0, h->stream>>>(h->v, first, in);
    else k_import_spins<<<grid_for(h->N, ny), 256, 0, h->stream>>>(h->v, first, in);
}

// ---- field ---------------------------------------------------------------------------------
void generate_field_host(rfim_pt* h, int d) {
    const uint32_t k0 = (uint32_t)(h->seeds[d] & 0xFFFFFFFFull), k1 = (uint32_t)(h->seeds[d] >> 32);
    int32_t* f = h->field_nat.data() + (long long)d * h->N;
    for (long long i = 0; i < h->N; ++i) {
        const Words4 w = philox4x32_10(k0, k1, (uint32_t)i, 0u, 0u, kDomField);
        if (h->kind == RFIM_FIELD_BIMODAL) {
            f[i] = (w.w0 >> 31) ? 1 : -1;
        } else {
            const double u1 = ((double)w.w0 + 1.0) / kTwo32;
            const double u2 = (double)w.w1 / kTwo32;
            const double radius = std::sqrt(-2.0 * std::log(u1));
            const double z = radius * std::cos((2.0 * M_PI) * u2);
            long long q = std::llrint(z * kFieldScale);
            q = std::min<long long>(std::max<long long>(q, -kFieldClamp), kFieldClamp);
            f[i] = (int32_t)q;
        }
    }
}

int upload_field(rfim_pt* h, int d) {
    const int L = h->L;
    const int32_t* f = h->field_nat.data() + (long long)d * h->N;
    const double hs = h->v.hs;
    if (h->kind == RFIM_FIELD_BIMODAL) {
        std::vector<uint8_t> fb(h->N);
        for (int z = 0; z < L; ++z) for (int y = 0; y < L; ++y) for (int x = 0; x < L; ++x) {
            int c; const long long j = layout_index(h, x, y, z, &c);
            fb[(long long)c * h->Nh + j] = f[x + (long long)L * (y + (long long)L * z)] > 0 ? 0x10 : 0x00;
        }
        CU(cudaMemcpyAsync(const_cast<uint8_t*>(h->v.fieldb) + (long long)d * h->N, fb.data(), h->N, cudaMemcpyHostToDevice, h->stream));
        if (h->fieldb_res) {
            std::vector<uint8_t> fr(h->N);
            for (int z = 0; z < L; ++z) for (int y = 0; y < L; ++y) for (int x = 0; x < L; ++x)
                fr[res_field_index(h, x, y, z)] = f[x + (long long)L * (y + (long long)L * z)] > 0 ? 0x80 : 0x00;
            CU(cudaMemcpyAsync(h->fieldb_res + (long long)d * h->N, fr.data(), h->N, cudaMemcpyHostToDevice, h->stream));
            CU(cudaStreamSynchronize(h->stream));         // fr goes out of scope
        }
        CU(cudaStreamSynchronize(h->stream));             // fb goes out of scope (a no-op after the one above)
        h->amax[d] = std::fabs(hs);
    } else {
        std::vector<float> fa(h->N);
        std::vector<int32_t> fg(h->N);
        double amax = 0.0;
        for (int z = 0; z < L; ++z) for (int y = 0; y < L; ++y) for (int x = 0; x < L; ++x) {
            int c; const long long j = layout_index(h, x, y, z, &c);
            const int32_t g = f[x + (long long)L * (y + (long long)L * z)];
            const double a = hs * (double)g;
            fa[(long long)c * h->Nh + j] = (float)g;              // |g| <= 2^23: exact
            fg[(long long)c * h->Nh + j] = g;
            amax = std::max(amax, std::fabs(a));
        }
        CU(cudaMemcpyAsync(const_cast<float*>(h->v.fielda) + (long long)d * h->N, fa.data(), h->N * sizeof(float), cudaMemcpyHostToDevice, h->stream));
        CU(cudaMemcpyAsync(const_cast<int32_t*>(h->v.fieldg) + (long long)d * h->N, fg.data(), h->N * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
        if (h->fielda_res) {
            std::vector<float> fr(h->N);
            for (int z = 0; z < L; ++z) for (int y = 0; y < L; ++y) for (int x = 0; x < L; ++x)
                fr[res_field_index(h, x, y, z)] = (float)f[x + (long long)L * (y + (long long)L * z)];
            CU(cudaMemcpyAsync(h->fielda_res + (long long)d * h->N, fr.data(), h->N * sizeof(float), cudaMemcpyHostToDevice, h->stream));
            std::vector<long long> gs(L, 0);
            for (int z = 0; z < L; ++z)
                for (long long i = 0; i < (long long)L * L; ++i) gs[z] += f[(long long)z * L * L + i];
            CU(cudaMemcpyAsync(h->gsum_res + (long long)d * L, gs.data(), (size_t)L * sizeof(long long), cudaMemcpyHostToDevice, h->stream));
            CU(cudaStreamSynchronize(h->stream));
        }
        CU(cudaStreamSynchronize(h->stream));
        h->amax[d] = amax;
    }
    return RFIM_OK;
}

// ---- acceptance tables (S3), binary64 on the host -----------------------------------
uint64_t threshold33(double x) {
    const double p = std::exp(-x);
    if (p >= 1.0) return (uint64_t)1 << 32;
    return (uint64_t)std::floor(p * kTwo32);
}

int upload_tables(rfim_pt* h) {
    const int R = h->R, n = h->n, D = h->D;
    std::vector<double> beta((size_t)D * R, 0.0);
    for (int d = 0; d < D; ++d)
        for (int t = 0; t < n; ++t) beta[(size_t)d * R + t] = 1.0 / h->T[(size_t)d * R + t];
    CU(cudaMemcpyAsync(const_cast<double*>(h->v.beta), beta.data(), beta.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    if (h->kind == RFIM_FIELD_BIMODAL) {
        std::vector<uint32_t> etab((size_t)D * R * 32, 0u), never((size_t)D * R, 0u);
        h->has_never = false;
        for (int d = 0; d < D; ++d)
            for (int t = 0; t < n; ++t) {
                const double b = beta[(size_t)d * R + t];
                uint32_t nv = 0;
                for (int idx = 0; idx < 32; ++idx) {
                    const int n1 = idx & 7, s = (idx >> 3) & 1, hb = (idx >> 4) & 1;
                    if (n1 == 7) { nv |= 1u << idx; continue; }              // unreachable neighbour count
                    const int k = s ? n1 : 6 - n1;                            // k = (s*n + 6)/2
                    const int bb = (s == hb) ? 1 : 0;                         // b = (s*h_i + 1)/2
                    const double dE = 2.0 * (h->J * (double)(2 * k - 6) + h->h * (double)(2 * bb - 1));
                    const uint64_t thr = threshold33(dE * b);
                    if (thr == 0) { nv |= 1u << idx; h->has_never = true; }
                    etab[((size_t)d * R + t) * 32 + idx] = (uint32_t)(thr - 1);
                }
                never[(size_t)d * R + t] = nv;
            }
        CU(cudaMemcpyAsync(const_cast<uint32_t*>(h->v.etab), etab.data(), etab.size() * 4, cudaMemcpyHostToDevice, h->stream));
        CU(cudaMemcpyAsync(const_cast<uint32_t*>(h->v.never), never.data(), never.size() * 4, cudaMemcpyHostToDevice, h->stream));
    } else {
        std::vector<GaussEntry> gtab((size_t)D * R * 16);
        std::vector<float> band((size_t)D * R, 0.f);
        for (int d = 0; d < D; ++d)
            for (int t = 0; t < n; ++t) {
                const double b = beta[(size_t)d * R + t];
                const double c = -2.0 * b * M_LOG2E;              // log2 P = c * sigma * (J n + hs g) ; +32 for the 2^32 scale
                for (int idx = 0; idx < 16; ++idx) {
                    const int n1 = idx & 7, s = (idx >> 3) & 1;
                    const double sigma = s ? 1.0 : -1.0;
                    GaussEntry e;
                    e.x = (float)(c * sigma * h->J * (double)(2 * n1 - 6) + 32.0);
                    e.y = (float)(c * sigma * h->v.hs);           // multiplies (float)g_i, which is exact
                    gtab[((size_t)d * R + t) * 16 + idx] = e;
                }
                // guard band: bound on |P~ - P| over the float path, in units of u.  arg = fl(g*fl(y) + fl(x)):
                // y's rounding moves it by <= |g y| 2^-24 <= aY 2^-24, x's by <= Xmax 2^-24, the fused multiply-add's one rounding by
                // <= 33 * 2^-24 wherever the decision is open (0 <= arg <= 33: below, P~ < 1 + band; above, both rules accept);
                // ex2.approx is taken at 2^-21 relative (twice its stated bound); float(u) is within 512 of u in either rounding
                // mode and the binary64 threshold within 1 of P 2^32.  The float decision can differ from the exact one only when
                // |float(u) - P~| <= 2^32 eta + 513: a quarter on top of that, and 1024 instead of 513.
                const double aY = h->amax[d] * std::fabs(c);
                const double Xmax = std::fabs(c) * std::fabs(h->J) * 6.0 + 32.0;
                const double arg_err = std::ldexp(aY + Xmax + 33.0, -24);
                const double eta = M_LN2 * arg_err + std::ldexp(1.0, -21);
                const double bd = 1.25 * eta * kTwo32 + 1024.0;
                band[(size_t)d * R + t] = (float)std::min(bd, 3.0e38);
            }
        CU(cudaMemcpyAsync(const_cast<GaussEntry*>(h->v.gtab), gtab.data(), gtab.size() * sizeof(GaussEntry), cudaMemcpyHostToDevice, h->stream));
        CU(cudaMemcpyAsync(const_cast<float*>(h->v.band), band.data(), band.size() * 4, cudaMemcpyHostToDevice, h->stream));
    }
    CU(cudaStreamSynchronize(h->stream));   // host vectors go out of scope
    return RFIM_OK;
}

int reset_statistics(rfim_pt* h) {
    const size_t DR = (size_t)h->D * h->R;
    CU(cudaMemsetAsync(h->v.att, 0, DR * 8, h->stream));
    CU(cudaMemsetAsync(h->v.accn, 0, DR * 8, h->stream));
    CU(cudaMemsetAsync(h->v.acc, 0, (size_t)h->D * h->acc_rows * 24, h->stream));
    h->series_steps = 0;
    return RFIM_OK;
}

int upload_permutation(rfim_pt* h, const std::vector<int32_t>& t2r) {   // [D][R], -1 beyond n
    std::vector<int32_t> r2t((size_t)h->D * h->R, -1);
    for (int d = 0; d < h->D; ++d)
        for (int t = 0; t < h->n; ++t) r2t[(size_t)d * h->R + t2r[(size_t)d * h->R + t]] = t;
    CU(cudaMemcpyAsync(h->v.t2r, t2r.data(), t2r.size() * 4, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->v.r2t, r2t.data(), r2t.size() * 4, cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int ensure_series(rfim_pt* h, long long rows) {
    if (rows <= h->series_cap) return RFIM_OK;
    long long cap = std::max<long long>(rows, h->series_cap * 2);
    cap = std::max<long long>(cap, 64);
    const size_t row_elems = (size_t)h->D * h->R * 3;
    long long* p = nullptr;
    int rc = alloc_into(h, &p, (size_t)cap * row_elems);
    if (rc) return rc;
    if (h->v.series && h->series_steps > 0)
        CU(cudaMemcpyAsync(p, h->v.series, (size_t)h->series_steps * row_elems * 8, cudaMemcpyDeviceToDevice, h->stream));
    if (h->v.series) { CU(cudaStreamSynchronize(h->stream)); release(h, h->v.series); }
    h->v.series = p;
    h->series_cap = cap;
    return RFIM_OK;
}

int ensure_stage(rfim_pt* h, size_t bytes) {
    if (bytes <= h->stage_bytes) return RFIM_OK;
    if (h->stage) { CU(cudaStreamSynchronize(h->stream)); release(h, h->stage); h->stage = nullptr; h->stage_bytes = 0; }
    int rc = alloc_into(h, &h->stage, bytes);
    if (rc) return rc;
    h->stage_bytes = bytes;
    return RFIM_OK;
}

// ---- launches ------------------------------------------------------------------------------
// kernel variants: 0 automatic, 1 site kernel, 2 word kernel, 3 flow kernel, 4 resident kernel (3, 4: L = 32 or 64),
// 5 small-lattice kernel (one CTA per replica, whole lattice in shared memory: L % 8 == 0, L^3 bytes resident)
bool flow_supported(const rfim_pt* h) { return h->L == 32 || h->L == 64; }

// the resident kernel's partition of the D*n*L planes over the grid, and whether the largest run fits in shared memory
// replicas one sweep of this handle visits: every active rank, or the active slots a shard stores (active slots are 0 .. n-1)
int iterated(const rfim_pt* h) {
    if (!h->shard) return h->n;
    // active slots are 0 .. n-1; the stored ones among them are the first ones of the window
    const int below = h->n - h->slot0;                        // slots slot0 + j * sstride < n  <=>  j < below / sstride (rounded up)
    if (below <= 0) return 0;
    return std::min(h->Rs, (below + h->sstride - 1) / h->sstride);
}

struct ResPlan { int grid, total, q, rem, cap_planes, cap_reps, nd, groups; size_t smem; bool ok; bool aligned; };
// plan for `nd` members per launch
ResPlan res_plan_nd(const rfim_pt* h, int nd) {
    ResPlan p{};
    p.ok = false;
    p.nd = nd; p.groups = (h->D + nd - 1) / nd;
    if (!flow_supported(h) || h->n < 1 || iterated(h) < 1 || h->sm_count < 1) return p;
    p.grid = std::min(h->sm_count, kResMaxGrid);
    if (h->res_grid_limit > 0) p.grid = std::min(p.grid, h->res_grid_limit);
    const long long nrep = (long long)nd * iterated(h);
    const long long total = nrep * h->L;
    if (total > (long long)p.grid * 32767) return p;
    p.total = (int)total;
    // Small problems (fewer than 2.5 replicas' worth of planes per CTA on average -- measured crossover at L = 32, see
    // profiles/r2_partition_scan.md): whole replicas per CTA instead of equal runs of planes.
    // A CTA then has no z-neighbour in another CTA at all -- no halo through L2, no progress words, no waiting on a
    // neighbour every phase -- and holds L planes' worth of tasks per phase instead of a handful; the price is that only
    // ceil(nrep / k) SMs work.  (this is also the regime each GPU of a replica split ends up in.)
    const int mode = h->res_partition;                      // 0 automatic, 1 equal runs, 2 replica-aligned
    const bool fits_whole = h->L <= res_max_planes(h->L);
    if (fits_whole && (mode == 2 || (mode == 0 && 2 * total < 5LL * p.grid * h->L))) {
        const int k = (int)((nrep + p.grid - 1) / p.grid);  // replicas per CTA
        if ((long long)k * h->L <= res_max_planes(h->L)) {
            p.aligned = true;
            p.q = k * h->L; p.rem = 0;
            p.grid = (int)((nrep + k - 1) / k);
            p.cap_planes = p.q;
            p.cap_reps = k;
            p.smem = res_smem_bytes(h->L, p.cap_reps);
            p.ok = p.smem <= (size_t)h->smem_optin;
            return p;
        }
    }
    p.q = p.total / p.grid; p.rem = p.total % p.grid;
    p.cap_planes = p.q + (p.rem ? 1 : 0);
    if (p.cap_planes > res_max_planes(h->L)) return p;
    p.cap_reps = (p.cap_planes + h->L - 2) / h->L + 1;
    if (p.cap_reps > 255) return p;
    p.smem = res_smem_bytes(h->L, p.cap_reps);
    p.ok = p.smem <= (size_t)h->smem_optin;
    return p;
}
// A batch whose planes do not all fit in the shared memory of the grid is swept in the fewest equal groups of members
// that do (members are independent; config 5 = 2 launches of 16 members).
ResPlan res_plan(const rfim_pt* h) {
    ResPlan p{};
    for (int groups = 1; groups <= h->D; ++groups) {
        const int nd = (h->D + groups - 1) / groups;
        if (groups > 1 && (h->D + nd - 1) / nd != groups) continue;
        p = res_plan_nd(h, nd);
        if (p.ok || groups >= 8) break;
    }
    return p;
}

bool small_supported(const rfim_pt* h) {
    return h->v.W > 0 && h->packing == 8 && small_smem_bytes(h->N) <= (size_t)h->smem_optin && (long long)h->D * h->R <= 65535;
}

int chosen_variant(const rfim_pt* h) {
    if (h->packing == 1) return 4;              // only the resident kernel reads the bit layout
    if (h->shard) return flow_supported(h) ? 4 : (small_supported(h) ? 5 : 4);   // kernels that visit a slot window
    if (h->variant != 0) return h->variant;
    if (res_plan(h).ok) return 4;
    if (flow_supported(h)) return 3;
    if (small_supported(h)) return 5;
    return h->v.W > 0 ? 2 : 1;
}

int launch_sweep(rfim_pt* h) {
    const int ny = h->D * h->n;
    const uint32_t g32 = (uint32_t)h->sweep_g;
    const bool word = chosen_variant(h) == 2;
    for (int colour = 0; colour < 2; ++colour) {
        if (word) k_sweep_word<<<grid_for(h->Nh / 4, ny), 256, 0, h->stream>>>(h->v, colour, g32);
        else k_sweep_site<<<grid_for(h->Nh, ny), 256, 0, h->stream>>>(h->v, colour, g32);
        h->launches += 1;
    }
    CU(cudaGetLastError());
    return RFIM_OK;
}

template <int KIND, int C, int CPT, bool NEVER>
int launch_flow_t(rfim_pt* h, const FlowParams& fp, long long items) {
    auto kernel = k_sweep_flow<KIND, C, CPT, NEVER>;
    long long blocks = max_coresident_blocks(kernel, kFlowThreads);
    if (blocks < 1) return fail(h, RFIM_ECUDA, "flow kernel does not fit on the device");
    blocks = std::min(blocks, items);
    CU(launch_cooperative(kernel, dim3((unsigned)blocks), dim3(kFlowThreads), h->stream, h->v, fp));
    h->launches += 1;
    return RFIM_OK;
}

// `sweeps` (<= 127) sweeps of every active replica in one persistent launch per <= 32 members
int launch_flow(rfim_pt* h, int sweeps) {
    const int C = h->L / 32, CPT = h->L == 64 ? 2 : 1;
    const int ZT = kFlowThreads * CPT / (h->L * C), S = h->L / ZT;
    for (int d0 = 0; d0 < h->D; d0 += kFlowMaxMembers) {
        FlowParams fp{};
        fp.RR = h->flow_rr;
        fp.G = (h->n + fp.RR - 1) / fp.RR;
        fp.d0 = d0;
        fp.nd = std::min(kFlowMaxMembers, h->D - d0);
        fp.phases = 2 * sweeps;
        fp.sweep0 = (uint32_t)h->sweep_g;
        fp.epoch = ++h->flow_epoch;
        fp.prog = h->flow_prog;
        fp.prog_stride_d = h->R * 32;
        fp.prog_stride_g = 32;
        fp.diag = h->v.diag;
        for (int dl = 0; dl < fp.nd; ++dl) {
            uint32_t k0 = (uint32_t)(h->seeds[d0 + dl] & 0xFFFFFFFFull), k1 = (uint32_t)(h->seeds[d0 + dl] >> 32);
            for (int r = 0; r < 10; ++r) { fp.rk[dl][2 * r] = k0; fp.rk[dl][2 * r + 1] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
        }
        const long long items = (long long)fp.phases * fp.nd * fp.G * S;
        int rc;
        if (h->kind == RFIM_FIELD_BIMODAL) {
            if (h->L == 64) rc = h->has_never ? launch_flow_t<0, 2, 2, true>(h, fp, items) : launch_flow_t<0, 2, 2, false>(h, fp, items);
            else rc = h->has_never ? launch_flow_t<0, 1, 1, true>(h, fp, items) : launch_flow_t<0, 1, 1, false>(h, fp, items);
        } else {
            if (h->L == 64) rc = launch_flow_t<1, 2, 2, false>(h, fp, items);
            else rc = launch_flow_t<1, 1, 1, false>(h, fp, items);
        }
        if (rc) return rc;
    }
    return RFIM_OK;
}

// the largest dynamic shared-memory size the kernel can be given on this device (opt-in maximum minus its static part)
cudaError_t set_max_dynamic_smem(const void* kernel, int optin) {
    cudaFuncAttributes fa{};
    cudaError_t e = cudaFuncGetAttributes(&fa, kernel);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
}

template <int KIND, int K, bool NEVER, bool UNI, bool MULTI = false>
int launch_res_t(rfim_pt* h, const ResPlan& pl, const ResParams& rp) {
    auto kernel = k_sweep_res<KIND, K, NEVER, UNI, kResThreads, MULTI>;
    // always the device's opt-in maximum, never this plan's own size: handles driven from several host threads share the
    // kernel's attribute, and a smaller value set by one between another's set and launch made that launch fail
    CU(set_max_dynamic_smem(reinterpret_cast<const void*>(kernel), h->smem_optin));
    void* argv[] = {const_cast<void*>(static_cast<const void*>(&h->v)), const_cast<void*>(static_cast<const void*>(&rp))};
    CU(cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(kernel), dim3((unsigned)pl.grid), dim3(kResThreads), argv, pl.smem, h->stream));
    h->launches += 1;
    return RFIM_OK;
}

template <int KIND, int K, bool NEVER>
int launch_res_u(rfim_pt* h, const ResPlan& pl, const ResParams& rp) {
    if (rp.nseg > 1) return launch_res_t<KIND, K, NEVER, true, true>(h, pl, rp);     // several moves per launch: single handles only
    return pl.nd == 1 ? launch_res_t<KIND, K, NEVER, true>(h, pl, rp) : launch_res_t<KIND, K, NEVER, false>(h, pl, rp);
}

template <int KIND, int K, bool NEVER>
int launch_res_k(rfim_pt* h, const ResPlan& pl, const ResParams& rp) { return launch_res_u<KIND, K, NEVER>(h, pl, rp); }

// How many sweeps the next launch of a persistent kernel covers and how many exchange steps it holds (pure: no handle).
// sweep_index = sweeps done so far, left = sweeps still asked for, k = exchange period (0: none), multi = the kernel may hold
// several steps (resident kernel, single handle).  A launch never exceeds 127 sweeps (the progress words carry 8 bits of phase),
// ends on an exchange step whenever it reaches one, and with `multi` runs on through as many whole periods as fit.
void plan_launch(uint64_t sweep_index, int64_t left, int k, bool multi, int64_t* chunk, int* nseg, int64_t* first) {
    *nseg = 1;
    *first = k > 0 ? (int64_t)k - (int64_t)(sweep_index % (uint64_t)k) : 0;
    *chunk = std::min<int64_t>(left, 127);
    if (k > 0) {
        if (multi && *chunk >= *first + k) {
            *nseg = 1 + (int)((*chunk - *first) / k);
            *chunk = *first + (int64_t)(*nseg - 1) * k;
        } else {
            *chunk = std::min<int64_t>(*chunk, *first);
        }
    }
}

// several parallel-tempering moves in one launch: single realisation, not sharded, exchange step fused
bool res_multi_ok(const rfim_pt* h) {
    if (!h->res_multi || h->shard || h->D != 1) return false;
    const ResPlan pl = res_plan(h);
    return pl.ok && pl.groups == 1 && pl.nd == 1;
}

// `sweeps` (<= 127) sweeps of every active replica of every member: one cooperative launch per group of members
// nseg > 1 (res_multi_moves() said so): the launch ends on an exchange step and holds nseg of them, the first after `first`
// sweeps, then every `period`; all of them run inside the kernel
int launch_res(rfim_pt* h, int sweeps, bool measure, bool* exchanged, int nseg = 1, int first = 0, int period = 0) {
    if (h->shard && iterated(h) == 0) { *exchanged = false; return RFIM_OK; }      // this shard stores no active slot
    const ResPlan pl0 = res_plan(h);
    if (!pl0.ok) return fail(h, RFIM_EINVAL, "resident kernel: the planes of one CTA do not fit in shared memory");
    *exchanged = measure && pl0.groups == 1 && h->D <= kResFusedExchangeMaxD && !h->shard;
    for (int d0 = 0; d0 < h->D; d0 += pl0.nd) {
        const int nd = std::min(pl0.nd, h->D - d0);
        const ResPlan pl = nd == pl0.nd ? pl0 : res_plan_nd(h, nd);
        if (!pl.ok) return fail(h, RFIM_EINVAL, "resident kernel: the last member group does not fit");
        ResParams rp{};
        rp.phases = 2 * sweeps;
        rp.measure = measure ? 1 : 0;
        rp.exchange = *exchanged ? 1 : 0;
        rp.nact = pl.q > 0 ? pl.grid : pl.rem;       // CTAs that own planes (a replica-aligned plan sizes the grid to them)
        rp.xstep = (uint32_t)h->xstep;
        rp.xrow = h->series_steps;
        rp.ticket = h->res_prog + kResMaxGrid;       // the word after the progress words (zeroed at create, left at zero)
        rp.xflag = h->res_prog + kResMaxGrid + 1;
        rp.nseg = nseg; rp.first2 = 2 * first; rp.period2 = 2 * period;
        rp.sweep0 = (uint32_t)h->sweep_g;
        rp.epoch = ++h->res_epoch;
        rp.prog = h->res_prog;
        rp.total_planes = pl.total; rp.q = pl.q; rp.rem = pl.rem;
        rp.cap_reps = pl.cap_reps;
        rp.d0 = d0;
        rp.fielda_res = h->fielda_res; rp.fieldb_res = h->fieldb_res; rp.gsum = h->gsum_res;
        rp.diag = h->v.diag;
        {
            uint32_t k0 = (uint32_t)(h->seeds[d0] & 0xFFFFFFFFull), k1 = (uint32_t)(h->seeds[d0] >> 32);
            for (int r = 0; r < 10; ++r) { rp.rk0[2 * r] = k0; rp.rk0[2 * r + 1] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
        }
        int rc;
        if (h->kind == RFIM_FIELD_BIMODAL) {
            if (h->L == 64) rc = h->has_never ? launch_res_k<0, 2, true>(h, pl, rp) : launch_res_k<0, 2, false>(h, pl, rp);
            else rc = h->has_never ? launch_res_k<0, 1, true>(h, pl, rp) : launch_res_k<0, 1, false>(h, pl, rp);
        } else {
            rc = h->L == 64 ? launch_res_k<1, 2, false>(h, pl, rp) : launch_res_k<1, 1, false>(h, pl, rp);
        }
        if (rc) return rc;
    }
    return RFIM_OK;
}

// `sweeps` (<= 127) sweeps of every active replica in ONE launch of the small-lattice kernel, with the measurement and (single
// handle, small batch) the exchange step inside
int small_threads(const rfim_pt* h) {
    const int words = (int)(h->Nh / 4);
    return std::min(kSmallMaxThreads, std::max(32, (words + 31) / 32 * 32));
}
// several moves per launch of the small-lattice kernel: the CTAs meet inside the launch, so all of them must be resident at once
// (a cooperative launch); unsharded handles whose exchange step is fused
bool small_multi_ok(rfim_pt* h) {
    if (!h->res_multi || h->shard || h->D > kResFusedExchangeMaxD || h->sm_count < 1) return false;
    const int nrep = h->D * iterated(h);
    if (h->small_per_sm < 0) {                          // CTAs of this handle's size one SM holds: a constant of the handle
        int per_sm = 0;
        const void* kern = h->kind == RFIM_FIELD_BIMODAL ? reinterpret_cast<const void*>(k_sweep_small<0, true>) : reinterpret_cast<const void*>(k_sweep_small<1, true>);
        if (set_max_dynamic_smem(kern, h->smem_optin) != cudaSuccess) return false;
        const cudaError_t e = h->kind == RFIM_FIELD_BIMODAL
            ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sweep_small<0, true>, small_threads(h), small_smem_bytes(h->N))
            : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sweep_small<1, true>, small_threads(h), small_smem_bytes(h->N));
        if (e != cudaSuccess) return false;
        h->small_per_sm = per_sm;
    }
    return nrep >= 1 && (long long)h->small_per_sm * h->sm_count >= nrep;
}

int launch_small(rfim_pt* h, int sweeps, bool measure, bool* exchanged, int nseg = 1, int first = 0, int period = 0) {
    *exchanged = false;
    const int nrep = h->D * iterated(h);
    if (nrep == 0) return RFIM_OK;                      // this shard stores no active slot
    SmallParams sp{};
    sp.phases = 2 * sweeps;
    sp.measure = measure ? 1 : 0;
    *exchanged = measure && h->D <= kResFusedExchangeMaxD && !h->shard;
    sp.exchange = *exchanged ? 1 : 0;
    sp.xstep = (uint32_t)h->xstep;
    sp.xrow = h->series_steps;
    sp.ticket = h->res_prog + kResMaxGrid;
    sp.sweep0 = (uint32_t)h->sweep_g;
    sp.nseg = nseg; sp.first2 = 2 * first; sp.period2 = 2 * period;
    sp.xflag = h->res_prog + kResMaxGrid + 1;
    sp.epoch = ++h->res_epoch;
    sp.diag = h->v.diag;
    const int threads = small_threads(h);
    const size_t smem = small_smem_bytes(h->N);
    const void* kern = nseg > 1 ? (h->kind == RFIM_FIELD_BIMODAL ? reinterpret_cast<const void*>(k_sweep_small<0, true>) : reinterpret_cast<const void*>(k_sweep_small<1, true>))
                                : (h->kind == RFIM_FIELD_BIMODAL ? reinterpret_cast<const void*>(k_sweep_small<0>) : reinterpret_cast<const void*>(k_sweep_small<1>));
    CU(set_max_dynamic_smem(kern, h->smem_optin));                     // (a constant: see launch_res_t)
    if (nseg > 1) {                                                    // the CTAs wait on one another: co-residency must be guaranteed
        void* argv[] = {const_cast<void*>(static_cast<const void*>(&h->v)), static_cast<void*>(&sp)};
        CU(cudaLaunchCooperativeKernel(kern, dim3((unsigned)nrep), dim3((unsigned)threads), argv, smem, h->stream));
    } else if (h->kind == RFIM_FIELD_BIMODAL) {
        k_sweep_small<0><<<nrep, threads, smem, h->stream>>>(h->v, sp);
    } else {
        k_sweep_small<1><<<nrep, threads, smem, h->stream>>>(h->v, sp);
    }
    h->launches += 1;
    CU(cudaGetLastError());
    return RFIM_OK;
}

// round-robin shard: slot s = j * G + r is row j of rank r
__global__ void k_terms_pack(const long long* __restrict__ acc, long long* __restrict__ all, int rank, int Rs, int G) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < Rs * 3) all[((long long)rank * Rs + i / 3) * 3 + i % 3] = acc[((long long)(i / 3) * G + rank) * 3 + i % 3];
}
__global__ void k_terms_unpack(long long* __restrict__ acc, const long long* __restrict__ all, int Rs, int G) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < G * Rs * 3) {
        const int c = i % 3, j = (i / 3) % Rs, r = i / (3 * Rs);
        acc[((long long)j * G + r) * 3 + c] = all[i];
    }
}

// replica shard: every rank now holds the energy terms of the slots it stores; the caller-supplied collective fills in
// the rows of the other ranks (an all-gather of 24 bytes per slot) so that every rank takes the same
// exchange decisions.  Runs on the handle's stream.
int gather_terms(rfim_pt* h) {
    if (!h->shard) return RFIM_OK;
    if (!h->gather && !h->nccl_comm) return fail(h, RFIM_ESTATE, "replica shard: no gather function set (rfim_pt_set_gather / rfim_pt_set_nccl)");
    constexpr int kNcclInt64 = 4;                               // ncclDataType_t
    if (h->nccl_comm) {
        // in-place all-gather (NCCL: sendbuff == recvbuff + rank * count) of Rs rows of 3 int64 per rank
        long long* buf = h->sstride == 1 ? h->v.acc : h->terms_all;
        if (h->sstride > 1) { k_terms_pack<<<(h->Rs * 3 + 127) / 128, 128, 0, h->stream>>>(h->v.acc, h->terms_all, h->rank, h->Rs, h->world); h->launches += 1; }
        if (h->nccl_all_gather(buf + (size_t)h->rank * h->Rs * 3, buf, (size_t)h->Rs * 3, kNcclInt64, h->nccl_comm, h->stream))
            return fail(h, RFIM_ECUDA, "replica shard: ncclAllGather failed");
        if (h->sstride > 1) { k_terms_unpack<<<(h->world * h->Rs * 3 + 127) / 128, 128, 0, h->stream>>>(h->v.acc, h->terms_all, h->Rs, h->world); h->launches += 1; }
        CU(cudaGetLastError());
        return RFIM_OK;
    }
    if (h->sstride == 1) {
        const int rc = h->gather(h->gather_user, h->v.acc, (size_t)h->slot0 * 24, (size_t)h->Rs * 24, h->acc_rows * 24, h->stream);
        if (rc) return fail(h, RFIM_ECUDA, "replica shard: the gather function failed");
        return RFIM_OK;
    }
    // round-robin deal: this rank's rows rank, rank + G, ... are gathered through a rank-major copy (contiguous per rank)
    const int cells = h->world * h->Rs * 3;
    k_terms_pack<<<(h->Rs * 3 + 127) / 128, 128, 0, h->stream>>>(h->v.acc, h->terms_all, h->rank, h->Rs, h->world);
    const int rc = h->gather(h->gather_user, h->terms_all, (size_t)h->rank * h->Rs * 24, (size_t)h->Rs * 24, (size_t)h->world * h->Rs * 24, h->stream);
    if (rc) return fail(h, RFIM_ECUDA, "replica shard: the gather function failed");
    k_terms_unpack<<<(cells + 127) / 128, 128, 0, h->stream>>>(h->v.acc, h->terms_all, h->Rs, h->world);
    h->launches += 2;
    CU(cudaGetLastError());
    return RFIM_OK;
}

int launch_reduce(rfim_pt* h) {
    View v = h->v;
    if (h->packing == 1) {
        // the stand-alone reduction reads the byte layout: unpack into scratch first (only the getters come here in
        // packed mode; the sweep path measures inside the resident kernel)
        const size_t DR = (size_t)h->D * h->Rs;
        if (!h->unpacked) { int rc = alloc_into(h, &h->unpacked, DR * (size_t)h->N); if (rc) return rc; }
        k_unpack_bits<<<grid_for((long long)(DR * (size_t)h->N / 8), 1), 256, 0, h->stream>>>(h->v.spins, h->unpacked, (long long)(DR * (size_t)h->N / 8));
        h->launches += 1;
        v.spins = h->unpacked; v.packed = 0;
    }
    if (v.W > 0) k_reduce_word<<<grid_for(h->Nh / 4, h->D * h->n), 256, 0, h->stream>>>(v);
    else k_reduce_site<<<grid_for(h->Nh, h->D * h->n), 256, 0, h->stream>>>(v);
    h->launches += 1;
    CU(cudaGetLastError());
    return RFIM_OK;
}

int launch_exchange(rfim_pt* h) {
    int threads = 32;
    while (threads < h->n && threads < 1024) threads *= 2;
    k_exchange<<<h->D, threads, 0, h->stream>>>(h->v, (uint32_t)h->xstep, h->series_steps, 1);
    h->launches += 1;
    CU(cudaGetLastError());
    return RFIM_OK;
}

int do_sweeps(rfim_pt* h, int64_t n_sweeps, int k) {
    if (!h->have_T) return fail(h, RFIM_ESTATE, "temperatures not set");
    if (n_sweeps < 0 || k < 0) return fail(h, RFIM_EINVAL, "negative argument");
    if (k > 0) {
        h->adapt_k = k;
        const long long steps = (long long)((h->sweep_g + (uint64_t)n_sweeps) / (uint64_t)k - h->sweep_g / (uint64_t)k);
        int rc = ensure_series(h, h->series_steps + steps);
        if (rc) return rc;
    }
    const int variant = chosen_variant(h);
    const bool flow = variant == 3 || variant == 4 || variant == 5;
    int64_t left = n_sweeps;
    while (left > 0) {
        int64_t chunk = 1, first = 0;
        int nseg = 1;
        // the resident kernel can hold several moves: as many whole exchange periods as fit in 127 sweeps
        if (flow) {
            // (the two *_multi_ok checks cost host time: ask only when the call does reach past the next exchange step)
            const bool spans = k > 0 && std::min<int64_t>(left, 127) >= (int64_t)k - (int64_t)(h->sweep_g % (uint64_t)k) + k;
            plan_launch(h->sweep_g, left, k, spans && ((variant == 4 && res_multi_ok(h)) || (variant == 5 && small_multi_ok(h))), &chunk, &nseg, &first);
        }
        // the resident kernel measures in the same launch when its chunk ends on an exchange step
        const bool step_after = k > 0 && ((h->sweep_g + (uint64_t)chunk) % (uint64_t)k) == 0;
        bool exchanged = false;
        int rc = variant == 4 ? launch_res(h, (int)chunk, step_after, &exchanged, nseg, (int)first, k)
               : variant == 5 ? launch_small(h, (int)chunk, step_after, &exchanged, nseg, (int)first, k)
               : (flow ? launch_flow(h, (int)chunk) : launch_sweep(h));
        if (rc) return rc;
        h->sweep_g += (uint64_t)chunk;
        left -= chunk;
        h->terms_fresh = step_after;                 // the lattices changed; an exchange step right now measures them
        if (step_after) {
            if (variant != 4 && variant != 5 && (rc = launch_reduce(h))) return rc;
            if ((rc = gather_terms(h))) return rc;
            if (!exchanged && (rc = launch_exchange(h))) return rc;
            h->series_steps += nseg;
            h->xstep += nseg;
        }
    }
    return RFIM_OK;
}

// current integer terms of every active replica, by rank: out [D][n][3]; also returns t2r [D][R]
// The persistent kernels give up a dependency wait after ~2^22 polls instead of hanging the GPU and set diag[0]:
// every synchronising getter reports that as an error (the lattices are then invalid).
int check_wait_flag(rfim_pt* h) {
    unsigned long long flag = 0;
    CU(cudaMemcpyAsync(&flag, h->v.diag, 8, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (flag != 0) return fail(h, RFIM_ESTATE, "a dependency wait of a persistent sweep kernel timed out: results are invalid");
    return RFIM_OK;
}

int measure_now(rfim_pt* h, std::vector<long long>& terms, std::vector<int32_t>& t2r) {
    const size_t DR = (size_t)h->D * h->R;
    std::vector<long long> acc(DR * 3);
    t2r.assign(DR, -1);
    int rc;
    if (h->terms_fresh) {
        // nothing has touched the lattices since the last exchange step measured them inside the sweep kernel: the terms
        // it consumed (kept by slot; an exchange moves temperatures, not lattices) are the terms of the current state
        CU(cudaMemcpyAsync(acc.data(), h->v.last, DR * 3 * 8, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(t2r.data(), h->v.t2r, DR * 4, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    } else {
        CU(cudaMemsetAsync(h->v.acc, 0, (size_t)h->D * h->acc_rows * 24, h->stream));
        rc = launch_reduce(h);
        if (rc) return rc;
        if ((rc = gather_terms(h))) return rc;
        CU(cudaMemcpyAsync(acc.data(), h->v.acc, DR * 3 * 8, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(t2r.data(), h->v.t2r, DR * 4, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemsetAsync(h->v.acc, 0, (size_t)h->D * h->acc_rows * 24, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    terms.assign((size_t)h->D * h->n * 3, 0);
    for (int d = 0; d < h->D; ++d)
        for (int t = 0; t < h->n; ++t) {
            const int slot = t2r[(size_t)d * h->R + t];
            for (int q = 0; q < 3; ++q) terms[((size_t)d * h->n + t) * 3 + q] = acc[((size_t)d * h->R + slot) * 3 + q];
        }
    return RFIM_OK;
}

int check_member(rfim_pt* h, int d) {
    if (!h) return RFIM_EINVAL;
    if (d < 0 || d >= h->D) return fail(h, RFIM_EINVAL, "member index out of range");
    return RFIM_OK;
}

int create_impl(rfim_pt** out, int L, int R, double J, double hh, int kind, int D, const uint64_t* seeds, int slot0 = 0, int nslots = -1, int sstride = 1) {
    if (!out) return RFIM_EINVAL;
    *out = nullptr;
    if (L < 2 || (L & 1) || L > 1024 || R < 1 || R > 4096 || D < 1 || D > 4096 || !seeds) return RFIM_EINVAL;
    if (kind != RFIM_FIELD_BIMODAL && kind != RFIM_FIELD_GAUSSIAN) return RFIM_EINVAL;
    if (!std::isfinite(J) || !std::isfinite(hh)) return RFIM_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return RFIM_ECUDA;   // no CPU fallback
    const bool shard = nslots >= 0;
    if (shard && (D != 1 || slot0 < 0 || nslots < 1 || slot0 >= R || sstride < 1)) return RFIM_EINVAL;
    if (shard && sstride == 1 && slot0 % nslots != 0) return RFIM_EINVAL;                       // contiguous windows, ordered by rank
    if (shard && sstride > 1 && (slot0 >= sstride || nslots != (R + sstride - 1) / sstride)) return RFIM_EINVAL;   // round-robin deal
    rfim_pt* h = new rfim_pt();
    h->L = L; h->R = R; h->D = D; h->kind = kind; h->J = J; h->h = hh;
    h->shard = shard; h->slot0 = shard ? slot0 : 0; h->Rs = shard ? nslots : R; h->sstride = shard ? sstride : 1;
    h->acc_rows = !shard ? (size_t)R : (sstride == 1 ? (size_t)((R + nslots - 1) / nslots) * nslots : (size_t)sstride * nslots);
    h->rank = !shard ? 0 : (sstride == 1 ? slot0 / nslots : slot0);
    h->world = !shard ? 1 : (sstride == 1 ? (int)(h->acc_rows / nslots) : sstride);
    h->N = (long long)L * L * L; h->Nh = h->N / 2;
    h->seeds.assign(seeds, seeds + D);
    h->field_nat.assign((size_t)D * h->N, 0);
    h->amax.assign(D, 0.0);
    h->T.assign((size_t)D * R, 0.0);
    View& v = h->v;
    v.L = L; v.Lh = L / 2; v.R = R; v.n = 0; v.D = D; v.kind = kind;
    v.W = (L % 8 == 0) ? L / 8 : 0;
    v.N = h->N; v.Nh = h->Nh;
    v.J = J; v.hs = (kind == RFIM_FIELD_BIMODAL) ? hh : hh / kFieldScale;
    v.shard = shard ? 1 : 0; v.slot0 = h->slot0; v.Rs = h->Rs; v.n_it = 0; v.sstride = h->sstride;
    const size_t DR = (size_t)D * R;
    int rc = RFIM_OK;
    auto A = [&](int r) { if (rc == RFIM_OK) rc = r; };
    A(alloc_into(h, &v.spins, (size_t)D * h->Rs * (size_t)h->N));
    if (kind == RFIM_FIELD_BIMODAL) {
        A(alloc_into(h, const_cast<uint8_t**>(&v.fieldb), (size_t)D * h->N));
        A(alloc_into(h, const_cast<uint32_t**>(&v.etab), DR * 32));
        A(alloc_into(h, const_cast<uint32_t**>(&v.never), DR));
    } else {
        A(alloc_into(h, const_cast<float**>(&v.fielda), (size_t)D * h->N));
        A(alloc_into(h, const_cast<int32_t**>(&v.fieldg), (size_t)D * h->N));
        A(alloc_into(h, const_cast<GaussEntry**>(&v.gtab), DR * 16));
        A(alloc_into(h, const_cast<float**>(&v.band), DR));
    }
    A(alloc_into(h, const_cast<double**>(&v.beta), DR));
    A(alloc_into(h, &v.t2r, DR));
    A(alloc_into(h, &v.r2t, DR));
    A(alloc_into(h, const_cast<uint32_t**>(&v.keys), (size_t)D * 2));
    A(alloc_into(h, &v.acc, (size_t)D * h->acc_rows * 3));
    if (h->sstride > 1) A(alloc_into(h, &h->terms_all, h->acc_rows * 3));
    A(alloc_into(h, &v.last, DR * 3));
    A(alloc_into(h, &v.ework, DR));
    A(alloc_into(h, &v.att, DR));
    A(alloc_into(h, &v.accn, DR));
    A(alloc_into(h, &v.diag, 4));
    A(alloc_into(h, &h->flow_prog, DR * 32));
    A(alloc_into(h, &h->res_prog, (size_t)kResMaxGrid + 2));
    if (flow_supported(h)) {
        if (kind == RFIM_FIELD_BIMODAL) A(alloc_into(h, &h->fieldb_res, (size_t)D * h->N));
        else { A(alloc_into(h, &h->fielda_res, (size_t)D * h->N)); A(alloc_into(h, &h->gsum_res, (size_t)D * L)); }
    }
    {
        int dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) {
            cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
            cudaDeviceGetAttribute(&h->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        }
    }
    if (rc != RFIM_OK) { rfim_pt_destroy(h); return rc; }
    auto body = [&]() -> int {
        std::vector<uint32_t> keys((size_t)D * 2);
        for (int d = 0; d < D; ++d) { keys[2 * d] = (uint32_t)(seeds[d] & 0xFFFFFFFFull); keys[2 * d + 1] = (uint32_t)(seeds[d] >> 32); }
        CU(cudaMemcpyAsync(const_cast<uint32_t*>(v.keys), keys.data(), keys.size() * 4, cudaMemcpyHostToDevice, h->stream));
        CU(cudaMemsetAsync(v.diag, 0, 32, h->stream));
        CU(cudaMemsetAsync(h->flow_prog, 0, DR * 32 * 4, h->stream));
        CU(cudaMemsetAsync(h->res_prog, 0, ((size_t)kResMaxGrid + 2) * 4, h->stream));
        CU(cudaMemsetAsync(v.t2r, 0xFF, DR * 4, h->stream));
        CU(cudaMemsetAsync(v.r2t, 0xFF, DR * 4, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        int r2 = reset_statistics(h);
        if (r2) return r2;
        for (int d = 0; d < D; ++d) {
            generate_field_host(h, d);
            if ((r2 = upload_field(h, d))) return r2;
        }
        k_init_spins<<<grid_for(h->N, D * h->Rs), 256, 0, h->stream>>>(v);
        h->launches += 1;
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(h->stream));
        return RFIM_OK;
    };
    rc = body();
    if (rc != RFIM_OK) { rfim_pt_destroy(h); return rc; }
    *out = h;
    return RFIM_OK;
}

// DESIGN.md S8: given the trial's rates, produce the new ladder for one member.
// Returns new temperatures, for each new rank the old rank it keeps the slot of (-1 = new replica),
// and for new replicas the old rank whose spins they copy.
struct AdaptPlan {
    std::vector<double> T;
    std::vector<int> keep_of;     // per new rank: old rank whose slot is kept, or -1
    std::vector<int> copy_of;     // per new rank: old rank copied (only where keep_of == -1)
};

AdaptPlan plan_adaptation(const std::vector<double>& T, const std::vector<double>& rate, int n, int R, int a_req) {
    AdaptPlan p;
    std::vector<int> order(n - 1);
    for (int t = 0; t < n - 1; ++t) order[t] = t;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return rate[x] < rate[y]; });
    std::vector<char> split(std::max(n - 1, 0), 0), removed(n, 0);
    if (n < R) {
        const int a = std::min(std::min(a_req, R - n), n - 1);
        for (int q = 0; q < a; ++q) split[order[q]] = 1;
    } else {
        const int a = std::min(a_req, n - 1);
        std::vector<char> inS(std::max(n - 1, 0), 0);
        for (int q = 0; q < a; ++q) inS[order[q]] = 1;
        const double rho = a > 0 ? rate[order[a - 1]] : 0.0;
        auto merged = [&](int u) { const double r1 = rate[u - 1], r2 = rate[u]; return (r1 * r2) * std::min(r1, r2); };
        std::vector<int> cand;
        for (int u = 1; u <= n - 2; ++u)
            if (!inS[u - 1] && !inS[u] && merged(u) > rho) cand.push_back(u);
        std::stable_sort(cand.begin(), cand.end(), [&](int x, int y) {
            if (merged(x) != merged(y)) return merged(x) > merged(y);
            return x > y;
        });
        int n_removed = 0;
        for (int u : cand) {
            if (n_removed == a) break;
            if (removed[u - 1] || removed[u + 1]) continue;
            removed[u] = 1;
            n_removed += 1;
        }
        for (int q = 0; q < n_removed; ++q) split[order[q]] = 1;
    }
    for (int t = 0; t < n; ++t) {
        if (!removed[t]) { p.T.push_back(T[t]); p.keep_of.push_back(t); p.copy_of.push_back(-1); }
        if (t < n - 1 && split[t]) { p.T.push_back((T[t] + T[t + 1]) / 2.0); p.keep_of.push_back(-1); p.copy_of.push_back(t); }
    }
    return p;
}

}  // namespace

// =================================================================================================
extern "C" {

int rfim_pt_set_allocator(rfim_pt_alloc_fn alloc, rfim_pt_free_fn release_fn) {
    if ((alloc == nullptr) != (release_fn == nullptr)) return RFIM_EINVAL;
    g_alloc = alloc; g_free = release_fn;
    return RFIM_OK;
}

int rfim_pt_create(rfim_pt** out, int L, int R, double J, double hh, int field_kind, uint64_t seed) {
    return create_impl(out, L, R, J, hh, field_kind, 1, &seed);
}

int rfim_pt_create_batch(rfim_pt** out, int L, int R, double J, double hh, int field_kind, int D, const uint64_t* seeds) {
    return create_impl(out, L, R, J, hh, field_kind, D, seeds);
}

int rfim_pt_create_shard(rfim_pt** out, int L, int R, double J, double hh, int field_kind, uint64_t seed, int slot0, int nslots) {
    return create_impl(out, L, R, J, hh, field_kind, 1, &seed, slot0, nslots);
}

int rfim_pt_create_shard_rr(rfim_pt** out, int L, int R, double J, double hh, int field_kind, uint64_t seed, int rank, int world) {
    if (world < 1 || rank < 0 || rank >= world || rank >= R) return RFIM_EINVAL;
    if (world == 1) return create_impl(out, L, R, J, hh, field_kind, 1, &seed, 0, R, 1);
    return create_impl(out, L, R, J, hh, field_kind, 1, &seed, rank, (R + world - 1) / world, world);
}

int rfim_pt_set_broadcast(rfim_pt* h, rfim_pt_bcast_fn fn, void* user) {
    if (!h) return RFIM_EINVAL;
    if (!h->shard) return fail(h, RFIM_EINVAL, "not a replica shard");
    h->bcast = fn; h->bcast_user = user;
    return RFIM_OK;
}

int rfim_pt_set_nccl(rfim_pt* h, void* comm, void* all_gather_fn, void* broadcast_fn) {
    if (!h) return RFIM_EINVAL;
    if (!h->shard) return fail(h, RFIM_EINVAL, "not a replica shard");
    if (comm && (!all_gather_fn || !broadcast_fn)) return fail(h, RFIM_EINVAL, "ncclAllGather and ncclBroadcast entry points are both needed");
    h->nccl_comm = comm;
    h->nccl_all_gather = reinterpret_cast<int (*)(const void*, void*, size_t, int, void*, cudaStream_t)>(all_gather_fn);
    h->nccl_broadcast = reinterpret_cast<int (*)(const void*, void*, size_t, int, int, void*, cudaStream_t)>(broadcast_fn);
    return RFIM_OK;
}

int rfim_pt_get_shard_layout(rfim_pt* h, int* rank, int* world, int* first_slot, int* stride, int* nslots) {
    if (!h) return RFIM_EINVAL;
    if (rank) *rank = h->rank;
    if (world) *world = h->world;
    if (first_slot) *first_slot = h->slot0;
    if (stride) *stride = h->sstride;
    if (nslots) *nslots = h->Rs;
    return RFIM_OK;
}

int rfim_pt_get_trial_rates(rfim_pt* h, int d, double* rate, int* n_pairs) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (h->trial_n < 2) return fail(h, RFIM_ESTATE, "no adaptation trial has run yet");
    if (n_pairs) *n_pairs = h->trial_n - 1;
    if (rate) std::memcpy(rate, h->trial_rates.data() + (size_t)d * h->R, (size_t)(h->trial_n - 1) * sizeof(double));
    return RFIM_OK;
}

int rfim_pt_set_gather(rfim_pt* h, rfim_pt_gather_fn fn, void* user) {
    if (!h) return RFIM_EINVAL;
    if (!h->shard) return fail(h, RFIM_EINVAL, "not a replica shard");
    h->gather = fn; h->gather_user = user;
    return RFIM_OK;
}

int rfim_pt_get_shard(rfim_pt* h, int* slot0, int* nslots, void** terms_device, size_t* terms_bytes) {
    if (!h) return RFIM_EINVAL;
    if (slot0) *slot0 = h->slot0;
    if (nslots) *nslots = h->Rs;
    if (terms_device) *terms_device = h->v.acc;
    if (terms_bytes) *terms_bytes = (size_t)h->D * h->acc_rows * 24;
    return RFIM_OK;
}

int rfim_pt_destroy(rfim_pt* h) {
    if (!h) return RFIM_OK;
    cudaStreamSynchronize(h->stream);
    for (void* p : h->owned) dev_free(p);
    delete h;
    return RFIM_OK;
}

const char* rfim_pt_last_error(rfim_pt* h) { return h ? h->err.c_str() : "null handle"; }

int rfim_pt_set_stream(rfim_pt* h, void* s) {
    if (!h) return RFIM_EINVAL;
    CU(cudaStreamSynchronize(h->stream));
    h->stream = reinterpret_cast<cudaStream_t>(s);
    return RFIM_OK;
}

int rfim_pt_synchronize(rfim_pt* h) {
    if (!h) return RFIM_EINVAL;
    return check_wait_flag(h);
}

int rfim_pt_set_packing(rfim_pt* h, int bits) {
    if (!h) return RFIM_EINVAL;
    if (bits != 8 && bits != 1) return fail(h, RFIM_EINVAL, "packing must be 8 (one byte per spin) or 1 (one bit per spin)");
    if (bits == h->packing) return RFIM_OK;
    const size_t DR = (size_t)h->D * h->Rs, nbits_bytes = DR * (size_t)h->N / 8;
    if (bits == 1) {
        if (h->variant != 0 && h->variant != 4) return fail(h, RFIM_EINVAL, "bit-packed storage is read by the resident kernel only (variant 0 or 4)");
        if (!flow_supported(h) || (h->have_T && !res_plan(h).ok))
            return fail(h, RFIM_EINVAL, "bit-packed storage needs the resident kernel (L = 32 or 64, planes resident in shared memory)");
        uint8_t* bitsbuf = nullptr;
        int rc = alloc_into(h, &bitsbuf, nbits_bytes);
        if (rc) return rc;
        k_pack_bits<<<grid_for((long long)nbits_bytes, 1), 256, 0, h->stream>>>(h->v.spins, bitsbuf, (long long)nbits_bytes);
        h->launches += 1;
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(h->stream));
        release(h, h->v.spins);
        h->v.spins = bitsbuf; h->v.packed = 1; h->packing = 1;
    } else {
        uint8_t* bytes = nullptr;
        int rc = alloc_into(h, &bytes, DR * (size_t)h->N);
        if (rc) return rc;
        k_unpack_bits<<<grid_for((long long)nbits_bytes, 1), 256, 0, h->stream>>>(h->v.spins, bytes, (long long)nbits_bytes);
        h->launches += 1;
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(h->stream));
        release(h, h->v.spins);
        if (h->unpacked) { release(h, h->unpacked); h->unpacked = nullptr; }
        h->v.spins = bytes; h->v.packed = 0; h->packing = 8;
    }
    return RFIM_OK;
}

int rfim_pt_set_kernel_variant(rfim_pt* h, int variant) {
    if (!h) return RFIM_EINVAL;
    if (variant < 0 || variant > 5) return fail(h, RFIM_EINVAL, "unknown kernel variant");
    if (variant == 5 && !small_supported(h)) return fail(h, RFIM_EINVAL, "small-lattice kernel needs L % 8 == 0 and L^3 bytes of shared memory");
    if (h->packing == 1 && variant != 0 && variant != 4) return fail(h, RFIM_EINVAL, "bit-packed storage is read by the resident kernel only");
    if (variant == 4 && !flow_supported(h)) return fail(h, RFIM_EINVAL, "resident kernel needs L = 32 or 64");
    if (variant == 2 && h->v.W == 0) return fail(h, RFIM_EINVAL, "word kernel needs L % 8 == 0");
    if (variant == 3 && !flow_supported(h)) return fail(h, RFIM_EINVAL, "flow kernel needs L = 32 or 64");
    h->variant = variant;
    return RFIM_OK;
}

int rfim_pt_set_tuning(rfim_pt* h, int key, int value) {
    if (!h) return RFIM_EINVAL;
    if (key == 0 && value >= 1 && value <= 64) { h->flow_rr = value; return RFIM_OK; }
    if (key == 1 && value >= 0 && value <= kResMaxGrid) { h->res_grid_limit = value; return RFIM_OK; }
    if (key == 2 && value >= 0 && value <= 2) { h->res_partition = value; return RFIM_OK; }
    if (key == 3 && value >= 0 && value <= 1) { h->res_multi = value; return RFIM_OK; }
    return fail(h, RFIM_EINVAL, "unknown tuning key or value out of range");
}

int rfim_pt_set_adapt_params(rfim_pt* h, int exchange_every, int insertions) {
    if (!h) return RFIM_EINVAL;
    if (exchange_every < 1 || insertions < 1) return fail(h, RFIM_EINVAL, "adapt parameters must be >= 1");
    h->adapt_k = exchange_every; h->adapt_a = insertions;
    return RFIM_OK;
}

int rfim_pt_set_temperatures(rfim_pt* h, const double* T, int n) {
    if (!h) return RFIM_EINVAL;
    if (!T || n < 1 || n > h->R) return fail(h, RFIM_EINVAL, "need 1 <= n <= R temperatures");
    for (int t = 0; t < n; ++t) {
        if (!(T[t] > 0.0) || !std::isfinite(T[t])) return fail(h, RFIM_EINVAL, "temperatures must be positive and finite");
        if (t > 0 && !(T[t] > T[t - 1])) return fail(h, RFIM_EINVAL, "temperatures must be strictly ascending");
    }
    h->n = n; h->v.n = n; h->v.n_it = iterated(h); h->terms_fresh = false;
    std::vector<int32_t> t2r((size_t)h->D * h->R, -1);
    for (int d = 0; d < h->D; ++d)
        for (int t = 0; t < n; ++t) { h->T[(size_t)d * h->R + t] = T[t]; t2r[(size_t)d * h->R + t] = t; }
    int rc;
    if ((rc = upload_permutation(h, t2r))) return rc;
    if ((rc = upload_tables(h))) return rc;
    if ((rc = reset_statistics(h))) return rc;
    h->have_T = true;
    return RFIM_OK;
}

int rfim_pt_sweep(rfim_pt* h, int64_t n_sweeps, int exchange_every) {
    if (!h) return RFIM_EINVAL;
    return do_sweeps(h, n_sweeps, exchange_every);
}

int rfim_pt_adapt_temperatures(rfim_pt* h, int64_t trial_sweeps) {
    if (!h) return RFIM_EINVAL;
    if (!h->have_T) return fail(h, RFIM_ESTATE, "temperatures not set");
    if (trial_sweeps < 0) return fail(h, RFIM_EINVAL, "negative argument");
    int rc;
    if ((rc = reset_statistics(h))) return rc;
    if ((rc = do_sweeps(h, trial_sweeps, h->adapt_k))) return rc;
    const int D = h->D, R = h->R, n = h->n;
    const size_t DR = (size_t)D * R;
    std::vector<unsigned long long> att(DR), acc(DR);
    std::vector<int32_t> t2r(DR);
    CU(cudaMemcpyAsync(att.data(), h->v.att, DR * 8, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaMemcpyAsync(acc.data(), h->v.accn, DR * 8, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaMemcpyAsync(t2r.data(), h->v.t2r, DR * 4, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    std::vector<AdaptPlan> plans(D);
    h->trial_rates.assign(DR, 0.0);
    h->trial_n = n;
    for (int d = 0; d < D; ++d) {
        std::vector<double> Td(h->T.begin() + (size_t)d * R, h->T.begin() + (size_t)d * R + n), rate(std::max(n - 1, 0));
        for (int t = 0; t < n - 1; ++t) {
            if (att[(size_t)d * R + t] == 0) return fail(h, RFIM_ESTATE, "a pair saw no exchange attempt in the trial");
            rate[t] = (double)acc[(size_t)d * R + t] / (double)att[(size_t)d * R + t];
            h->trial_rates[(size_t)d * R + t] = rate[t];
        }
        plans[d] = plan_adaptation(Td, rate, n, R, h->adapt_a);
        if (plans[d].T.size() != plans[0].T.size()) return fail(h, RFIM_ESTATE, "members disagree on the new replica count");
    }
    const int n_new = (int)plans[0].T.size();
    std::vector<int32_t> new_t2r(DR, -1);
    for (int d = 0; d < D; ++d) {
        int next_slot = n;                         // pool slots n..R-1
        for (int j = 0; j < n_new; ++j) {
            const AdaptPlan& p = plans[d];
            int slot;
            if (n_new == n) {
                slot = t2r[(size_t)d * R + j];     // fixed count: the slot at rank j keeps rank j
            } else if (p.keep_of[j] >= 0) {
                slot = t2r[(size_t)d * R + p.keep_of[j]];
            } else {
                slot = next_slot++;
                const int src = t2r[(size_t)d * R + p.copy_of[j]];
                if (h->shard) {
                    // the new replica lives on the rank its pool slot belongs to (slot mod G for a round-robin
                    // deal); its spins come from the rank that stores the colder neighbour: one broadcast of N/8 bytes
                    if (!h->bcast && !h->nccl_comm) return fail(h, RFIM_ESTATE, "replica shard: inserting a replica needs the lattice broadcast (rfim_pt_set_broadcast / rfim_pt_set_nccl)");
                    if ((rc = ensure_stage(h, (size_t)h->N / 8))) return rc;
                    uint8_t* buf = reinterpret_cast<uint8_t*>(h->stage);
                    if (h->v.stores(src)) { launch_export_bits(h, 1, h->v.stored_index(src), buf); h->launches += 1; }
                    const int root = h->sstride == 1 ? src / h->Rs : src % h->world;
                    const int brc = h->nccl_comm ? h->nccl_broadcast(buf, buf, (size_t)h->N / 8, /* ncclUint8 */ 1, root, h->nccl_comm, h->stream)
                                                 : h->bcast(h->bcast_user, buf, (size_t)h->N / 8, root, h->stream);
                    if (brc) return fail(h, RFIM_ECUDA, "replica shard: the lattice broadcast failed");
                    if (h->v.stores(slot)) { launch_import_bits(h, 1, h->v.stored_index(slot), buf); h->launches += 1; }
                    CU(cudaGetLastError());
                } else {
                    const size_t lat = (size_t)h->N / (h->packing == 1 ? 8 : 1);      // bytes per lattice
                    CU(cudaMemcpyAsync(h->v.spins + ((size_t)d * R + slot) * lat, h->v.spins + ((size_t)d * R + src) * lat,
                                       lat, cudaMemcpyDeviceToDevice, h->stream));
                }
            }
            new_t2r[(size_t)d * R + j] = slot;
            h->T[(size_t)d * R + j] = p.T[j];
        }
    }
    h->n = n_new; h->v.n = n_new; h->v.n_it = iterated(h); h->terms_fresh = false;
    if ((rc = upload_permutation(h, new_t2r))) return rc;
    if ((rc = upload_tables(h))) return rc;
    if ((rc = reset_statistics(h))) return rc;
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int rfim_pt_observables(rfim_pt* h, double* E, double* M, double* rate) {
    if (!h) return RFIM_EINVAL;
    if (!h->have_T) return fail(h, RFIM_ESTATE, "temperatures not set");
    std::vector<long long> terms; std::vector<int32_t> t2r;
    int rc = measure_now(h, terms, t2r);
    if (rc) return rc;
    if ((rc = check_wait_flag(h))) return rc;
    const int D = h->D, n = h->n, R = h->R;
    for (int d = 0; d < D; ++d)
        for (int t = 0; t < n; ++t) {
            const long long* q = &terms[((size_t)d * n + t) * 3];
            if (E) E[(size_t)d * n + t] = (-h->J * (double)q[0]) - (h->v.hs * (double)q[1]);
            if (M) M[(size_t)d * n + t] = (double)q[2] / (double)h->N;
        }
    if (rate) {
        const size_t DR = (size_t)D * R;
        std::vector<unsigned long long> att(DR), acc(DR);
        CU(cudaMemcpyAsync(att.data(), h->v.att, DR * 8, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(acc.data(), h->v.accn, DR * 8, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        for (int d = 0; d < D; ++d)
            for (int t = 0; t < n - 1; ++t)
                rate[(size_t)d * (n - 1) + t] = att[(size_t)d * R + t] ? (double)acc[(size_t)d * R + t] / (double)att[(size_t)d * R + t] : -1.0;
    }
    return RFIM_OK;
}

int rfim_pt_get_info(rfim_pt* h, int* L, int* R, int* n, int* D, int* kind) {
    if (!h) return RFIM_EINVAL;
    if (L) *L = h->L; if (R) *R = h->R; if (n) *n = h->n; if (D) *D = h->D; if (kind) *kind = h->kind;
    return RFIM_OK;
}

int rfim_pt_get_spins_slot(rfim_pt* h, int d, int slot, int8_t* out) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (slot < 0 || slot >= h->R || !out) return fail(h, RFIM_EINVAL, "bad slot or null buffer");
    if (!h->v.stores(slot)) return fail(h, RFIM_EINVAL, "replica shard: this rank does not store that slot");
    if ((rc = ensure_stage(h, (size_t)h->N))) return rc;
    launch_export_spins(h, 1, d * h->Rs + h->v.stored_index(slot), h->stage);
    h->launches += 1;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(out, h->stage, (size_t)h->N, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int rfim_pt_get_spins_member(rfim_pt* h, int d, int temp_rank, int8_t* out) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (!h->have_T) return fail(h, RFIM_ESTATE, "temperatures not set");
    if (temp_rank < 0 || temp_rank >= h->n) return fail(h, RFIM_EINVAL, "temperature rank out of range");
    int32_t slot = -1;
    CU(cudaMemcpyAsync(&slot, h->v.t2r + (size_t)d * h->R + temp_rank, 4, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return rfim_pt_get_spins_slot(h, d, slot, out);
}

int rfim_pt_get_spins(rfim_pt* h, int temp_rank, int8_t* out) { return rfim_pt_get_spins_member(h, 0, temp_rank, out); }

int rfim_pt_set_spins_slot(rfim_pt* h, int d, int slot, const int8_t* in) {
    if (h) h->terms_fresh = false;
    int rc = check_member(h, d);
    if (rc) return rc;
    if (slot < 0 || slot >= h->R || !in) return fail(h, RFIM_EINVAL, "bad slot or null buffer");
    for (long long i = 0; i < h->N; ++i)
        if (in[i] != 1 && in[i] != -1) return fail(h, RFIM_EINVAL, "spins must be +1 or -1");
    if (!h->v.stores(slot)) return fail(h, RFIM_EINVAL, "replica shard: this rank does not store that slot");
    if ((rc = ensure_stage(h, (size_t)h->N))) return rc;
    CU(cudaMemcpyAsync(h->stage, in, (size_t)h->N, cudaMemcpyHostToDevice, h->stream));
    launch_import_spins(h, 1, d * h->Rs + h->v.stored_index(slot), h->stage);
    h->launches += 1;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int rfim_pt_get_spins_all(rfim_pt* h, int8_t* out) {
    if (!h || !out) return RFIM_EINVAL;
    const int DR = h->D * h->Rs;          // every stored lattice (a replica shard: its slot window)
    int rc = ensure_stage(h, (size_t)DR * h->N);
    if (rc) return rc;
    launch_export_spins(h, DR, 0, h->stage);
    h->launches += 1;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(out, h->stage, (size_t)DR * h->N, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int rfim_pt_set_spins_all(rfim_pt* h, const int8_t* in) {
    if (h) h->terms_fresh = false;
    if (!h || !in) return RFIM_EINVAL;
    const int DR = h->D * h->Rs;
    int rc = ensure_stage(h, (size_t)DR * h->N);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->stage, in, (size_t)DR * h->N, cudaMemcpyHostToDevice, h->stream));
    launch_import_spins(h, DR, 0, h->stage);
    h->launches += 1;
    CU(cudaGetLastError());
    return RFIM_OK;
}

int rfim_pt_get_spins_all_bits(rfim_pt* h, uint8_t* out) {
    if (!h || !out) return RFIM_EINVAL;
    const int DR = h->D * h->Rs;
    const size_t bytes = (size_t)DR * (size_t)(h->N / 8);
    int rc = ensure_stage(h, bytes);
    if (rc) return rc;
    launch_export_bits(h, DR, 0, reinterpret_cast<uint8_t*>(h->stage));
    h->launches += 1;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(out, h->stage, bytes, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int rfim_pt_set_spins_all_bits(rfim_pt* h, const uint8_t* in) {
    if (h) h->terms_fresh = false;
    if (!h || !in) return RFIM_EINVAL;
    const int DR = h->D * h->Rs;
    const size_t bytes = (size_t)DR * (size_t)(h->N / 8);
    int rc = ensure_stage(h, bytes);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->stage, in, bytes, cudaMemcpyHostToDevice, h->stream));
    launch_import_bits(h, DR, 0, reinterpret_cast<const uint8_t*>(h->stage));
    h->launches += 1;
    CU(cudaGetLastError());
    return RFIM_OK;
}

int rfim_pt_get_field(rfim_pt* h, int d, int32_t* out) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (!out) return fail(h, RFIM_EINVAL, "null buffer");
    std::memcpy(out, h->field_nat.data() + (size_t)d * h->N, (size_t)h->N * 4);
    return RFIM_OK;
}

int rfim_pt_set_field(rfim_pt* h, int d, const int32_t* in) {
    if (h) h->terms_fresh = false;
    int rc = check_member(h, d);
    if (rc) return rc;
    if (!in) return fail(h, RFIM_EINVAL, "null buffer");
    for (long long i = 0; i < h->N; ++i) {
        if (h->kind == RFIM_FIELD_BIMODAL) { if (in[i] != 1 && in[i] != -1) return fail(h, RFIM_EINVAL, "bimodal field must be +-1"); }
        else if (in[i] > kFieldClamp || in[i] < -kFieldClamp) return fail(h, RFIM_EINVAL, "Gaussian field out of range");
    }
    CU(cudaStreamSynchronize(h->stream));
    std::memcpy(h->field_nat.data() + (size_t)d * h->N, in, (size_t)h->N * 4);
    if ((rc = upload_field(h, d))) return rc;
    if (h->have_T && (rc = upload_tables(h))) return rc;     // the guard band depends on max |a_i|
    return RFIM_OK;
}

int rfim_pt_get_permutation(rfim_pt* h, int d, int32_t* t2r) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (!t2r) return fail(h, RFIM_EINVAL, "null buffer");
    CU(cudaMemcpyAsync(t2r, h->v.t2r + (size_t)d * h->R, (size_t)h->n * 4, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int rfim_pt_set_permutation(rfim_pt* h, int d, const int32_t* t2r_in) {
    if (h) h->terms_fresh = false;
    int rc = check_member(h, d);
    if (rc) return rc;
    if (!t2r_in || !h->have_T) return fail(h, RFIM_EINVAL, "null buffer or temperatures not set");
    const size_t DR = (size_t)h->D * h->R;
    std::vector<int32_t> t2r(DR);
    CU(cudaMemcpyAsync(t2r.data(), h->v.t2r, DR * 4, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    std::vector<char> seen(h->R, 0);
    for (int t = 0; t < h->n; ++t) {
        const int s = t2r_in[t];
        if (s < 0 || s >= h->R || seen[s]) return fail(h, RFIM_EINVAL, "not a permutation of slots");
        seen[s] = 1;
        t2r[(size_t)d * h->R + t] = s;
    }
    return upload_permutation(h, t2r);
}

int rfim_pt_get_temperatures(rfim_pt* h, int d, double* T, int* n) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (n) *n = h->n;
    if (T) for (int t = 0; t < h->n; ++t) T[t] = h->T[(size_t)d * h->R + t];
    return RFIM_OK;
}

int rfim_pt_get_counters(rfim_pt* h, uint64_t* sweep_index, uint64_t* exchange_step) {
    if (!h) return RFIM_EINVAL;
    if (sweep_index) *sweep_index = h->sweep_g;
    if (exchange_step) *exchange_step = h->xstep;
    return RFIM_OK;
}

int rfim_pt_set_counters(rfim_pt* h, uint64_t sweep_index, uint64_t exchange_step) {
    if (!h) return RFIM_EINVAL;
    h->sweep_g = sweep_index; h->xstep = exchange_step;
    return RFIM_OK;
}

int rfim_pt_get_energy_terms(rfim_pt* h, int d, int64_t* Eb, int64_t* Ef, int64_t* Msum) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (!h->have_T) return fail(h, RFIM_ESTATE, "temperatures not set");
    std::vector<long long> terms; std::vector<int32_t> t2r;
    if ((rc = measure_now(h, terms, t2r))) return rc;
    for (int t = 0; t < h->n; ++t) {
        const long long* q = &terms[((size_t)d * h->n + t) * 3];
        if (Eb) Eb[t] = q[0]; if (Ef) Ef[t] = q[1]; if (Msum) Msum[t] = q[2];
    }
    return RFIM_OK;
}

int64_t rfim_pt_timeseries_steps(rfim_pt* h) { return h ? h->series_steps : 0; }

int rfim_pt_get_timeseries(rfim_pt* h, int d, int64_t* Eb, int64_t* Ef, int64_t* Msum) {
    int rc = check_member(h, d);
    if (rc) return rc;
    const long long steps = h->series_steps;
    if (steps == 0) return RFIM_OK;
    const size_t row = (size_t)h->D * h->R * 3;
    std::vector<long long> buf((size_t)steps * row);
    CU(cudaMemcpyAsync(buf.data(), h->v.series, buf.size() * 8, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    for (long long s = 0; s < steps; ++s)
        for (int t = 0; t < h->n; ++t) {
            const long long* q = &buf[(size_t)s * row + ((size_t)d * h->R + t) * 3];
            if (Eb) Eb[s * h->n + t] = q[0]; if (Ef) Ef[s * h->n + t] = q[1]; if (Msum) Msum[s * h->n + t] = q[2];
        }
    return RFIM_OK;
}

namespace {
// [D][n][5] thermal moments of the series over steps [skip, steps), computed on the device
int thermal_moments_all(rfim_pt* h, int64_t skip, std::vector<double>& mom) {
    if (!h->have_T) return fail(h, RFIM_ESTATE, "temperatures not set");
    if (skip < 0 || skip >= h->series_steps) return fail(h, RFIM_ESTATE, "no measurement steps after `skip` (sweep with exchange_every > 0 first)");
    const size_t cnt = (size_t)h->D * h->n * 5;
    if (!h->moments_dev) {                              // [D][R][5], allocated on first use, released with the handle
        int rc = alloc_into(h, &h->moments_dev, (size_t)h->D * h->R * 5);
        if (rc) return rc;
    }
    k_thermal_moments<<<h->D * h->n, 256, 0, h->stream>>>(h->v, (long long)skip, h->series_steps, h->moments_dev);
    h->launches += 1;
    mom.assign(cnt, 0.0);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(mom.data(), h->moments_dev, cnt * 8, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}
}  // namespace

int rfim_pt_thermal_moments(rfim_pt* h, int d, int64_t skip, double* out) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (!out) return fail(h, RFIM_EINVAL, "null buffer");
    std::vector<double> mom;
    if ((rc = thermal_moments_all(h, skip, mom))) return rc;
    std::memcpy(out, mom.data() + (size_t)d * h->n * 5, (size_t)h->n * 5 * 8);
    return RFIM_OK;
}

int rfim_pt_thermal_observables(rfim_pt* h, int64_t skip, double* absM, double* C, double* g) {
    if (!h) return RFIM_EINVAL;
    std::vector<double> mom;
    int rc = thermal_moments_all(h, skip, mom);
    if (rc) return rc;
    const int D = h->D, n = h->n;
    for (int t = 0; t < n; ++t) {
        double sa = 0, sc = 0, s2 = 0, s4 = 0;
        for (int d = 0; d < D; ++d) {
            const double* m = mom.data() + ((size_t)d * n + t) * 5;
            const double T = h->T[(size_t)d * h->R + t];
            sa += m[2];
            sc += ((double)h->N / (T * T)) * (m[1] - m[0] * m[0]);      // Eq. 12 per realisation
            s2 += m[3]; s4 += m[4];
        }
        const double m2 = s2 / D, m4 = s4 / D;
        if (absM) absM[t] = sa / D;                                     // Eq. 11
        if (C) C[t] = sc / D;
        if (g) g[t] = 0.5 * (3.0 - m4 / (m2 * m2));                     // Eq. 13: ratio of the disorder averages
    }
    return RFIM_OK;
}

int rfim_pt_get_exchange_counts(rfim_pt* h, int d, uint64_t* attempted, uint64_t* accepted) {
    int rc = check_member(h, d);
    if (rc) return rc;
    const int m = std::max(h->n - 1, 0);
    if (attempted) CU(cudaMemcpyAsync(attempted, h->v.att + (size_t)d * h->R, (size_t)m * 8, cudaMemcpyDeviceToHost, h->stream));
    if (accepted) CU(cudaMemcpyAsync(accepted, h->v.accn + (size_t)d * h->R, (size_t)m * 8, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return RFIM_OK;
}

int rfim_pt_get_bimodal_threshold(rfim_pt* h, int d, int rank, int k, int b, uint64_t* thr) {
    int rc = check_member(h, d);
    if (rc) return rc;
    if (h->kind != RFIM_FIELD_BIMODAL || !h->have_T || rank < 0 || rank >= h->n || k < 0 || k > 6 || b < 0 || b > 1 || !thr)
        return fail(h, RFIM_EINVAL, "bad threshold query");
    // device index for s = +1: n1 = k, hb = b (s = +1 so b = hb)
    const int idx = k | (1 << 3) | (b << 4);
    uint32_t e = 0, nv = 0;
    CU(cudaMemcpyAsync(&e, h->v.etab + ((size_t)d * h->R + rank) * 32 + idx, 4, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaMemcpyAsync(&nv, h->v.never + (size_t)d * h->R + rank, 4, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    *thr = ((nv >> idx) & 1u) ? 0ull : (uint64_t)e + 1ull;
    return RFIM_OK;
}

int rfim_pt_plan_launch(uint64_t sweep_index, int64_t n_sweeps, int exchange_every, int several_moves, int64_t* launch_sweeps,
                        int* exchange_steps) {
    if (n_sweeps < 1 || exchange_every < 0 || !launch_sweeps || !exchange_steps) return RFIM_EINVAL;
    int64_t first = 0;
    int nseg = 1;
    plan_launch(sweep_index, n_sweeps, exchange_every, several_moves != 0, launch_sweeps, &nseg, &first);
    *exchange_steps = (exchange_every > 0 && (sweep_index + (uint64_t)*launch_sweeps) % (uint64_t)exchange_every == 0) ? nseg : 0;
    return RFIM_OK;
}

int rfim_pt_plan_adaptation(const double* T, const double* rate, int n, int R, int a, double* out_T, int* out_n) {
    if (!T || !rate || !out_T || !out_n || n < 2 || n > R || a < 0) return RFIM_EINVAL;
    const std::vector<double> Tv(T, T + n), rv(rate, rate + n - 1);
    const AdaptPlan plan = plan_adaptation(Tv, rv, n, R, a);
    if ((int)plan.T.size() > R) return RFIM_EINVAL;
    for (size_t i = 0; i < plan.T.size(); ++i) out_T[i] = plan.T[i];
    *out_n = (int)plan.T.size();
    return RFIM_OK;
}

int rfim_pt_get_diagnostics(rfim_pt* h, uint64_t diag[4]) {
    if (!h || !diag) return RFIM_EINVAL;
    unsigned long long d4[4];
    CU(cudaMemcpyAsync(d4, h->v.diag, 32, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    if (d4[0] != 0) return fail(h, RFIM_ESTATE, "a dependency wait of a persistent sweep kernel timed out: results are invalid");
    diag[0] = h->launches; diag[1] = d4[1]; diag[2] = d4[2]; diag[3] = d4[3];
    return RFIM_OK;
}

}  // extern "C"

// ---- roofline microbenchmarks ---------------------------------------------------------------------
namespace {

// Philox4x32-10 alone, with the sweep's own counter layout (S2): c0 = word index (varies per call), c1 = sweep,
// c2 = slot, c3 = domain (warp-uniform), round keys from the constant bank; four independent calls in flight per
// thread.  The compiler hoists the warp-uniform part of the first two rounds exactly as it does in the sweep kernels,
// so this is the tightest Philox-only bound for this method: ~18 wide multiplies + ~18 three-input XORs per call.
struct BenchKeys { uint32_t k[20]; };
__global__ void __launch_bounds__(256) k_bench_philox(uint32_t* out, int calls, BenchKeys rk, uint32_t sweep, uint32_t slot) {
    constexpr int ILP = 4;
    uint32_t acc = 0, base = (blockIdx.x * blockDim.x + threadIdx.x) * ILP;
    for (int i = 0; i < calls; i += ILP) {
        uint32_t c0[ILP], c1[ILP], c2[ILP], c3[ILP];
#pragma unroll
        for (int j = 0; j < ILP; ++j) { c0[j] = base + j; c1[j] = sweep; c2[j] = slot; c3[j] = kDomColour0; }
#pragma unroll
        for (int r = 0; r < 10; ++r) {
#pragma unroll
            for (int j = 0; j < ILP; ++j) {
                const uint32_t hi0 = __umulhi(kPhiloxM0, c0[j]), lo0 = kPhiloxM0 * c0[j];
                const uint32_t hi1 = __umulhi(kPhiloxM1, c2[j]), lo1 = kPhiloxM1 * c2[j];
                const uint32_t n0 = hi1 ^ c1[j] ^ rk.k[2 * r], n2 = hi0 ^ c3[j] ^ rk.k[2 * r + 1];
                c1[j] = lo1; c3[j] = lo0; c0[j] = n0; c2[j] = n2;
            }
        }
#pragma unroll
        for (int j = 0; j < ILP; ++j) acc ^= c0[j] ^ c1[j] ^ c2[j] ^ c3[j];
        base += gridDim.x * blockDim.x * ILP;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// Issue-cost probe ("what an instruction costs next to Philox"): the same Philox stream with N extra
// instructions of ONE kind per call, spread between the rounds, on operands that form their own dependency chains.  The
// slope of the time per warp-row against N / 4 is what one more warp instruction of that kind costs the sub-partition
// while it runs the Philox stream: the quantity the row update has to minimise.
enum { kProbeNone = 0, kProbeLop3 = 1, kProbePrmt = 2, kProbeI2fp = 3, kProbeI2fRm = 4, kProbeFfma = 5, kProbeFadd = 6, kProbeMufu = 7, kProbeLds64 = 8, kProbeKinds = 9 };
template <int OP>
__device__ __forceinline__ void probe_op(uint32_t (&a)[4], float (&f)[4], int j, uint32_t saddr) {
    uint32_t& x = a[j & 3]; const uint32_t y = a[(j + 1) & 3];
    float& fx = f[j & 3]; const float fy = f[(j + 1) & 3];
    if (OP == kProbeLop3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(y), "r"(a[(j + 2) & 3]));
    if (OP == kProbePrmt) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(x) : "r"(y), "r"(a[(j + 2) & 3]));
    if (OP == kProbeI2fp) asm volatile("{ .reg .f32 t; cvt.rn.f32.u32 t, %1; mov.b32 %0, t; }" : "=r"(x) : "r"(y));
    if (OP == kProbeI2fRm) asm volatile("{ .reg .f32 t; cvt.rm.f32.u32 t, %1; mov.b32 %0, t; }" : "=r"(x) : "r"(y));
    if (OP == kProbeFfma) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fx) : "f"(fy), "f"(f[(j + 2) & 3]));
    if (OP == kProbeFadd) asm volatile("add.f32 %0, %0, %1;" : "+f"(fx) : "f"(fy));
    if (OP == kProbeMufu) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(fx));
    if (OP == kProbeLds64) { uint32_t r0, r1; asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r0), "=r"(r1) : "r"(saddr + (uint32_t)(j & 15) * 256u)); x ^= r0; a[(j + 3) & 3] = r1; }
}
template <int OP, int N>
__global__ void __launch_bounds__(512, 1) k_bench_issue(uint32_t* out, int iters, BenchKeys rk, uint32_t sweep, uint32_t slot) {
    extern __shared__ __align__(16) uint8_t probe_smem[];
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) reinterpret_cast<uint32_t*>(probe_smem)[i] = i * 2654435761u;
    __syncthreads();
    const uint32_t saddr = (uint32_t)__cvta_generic_to_shared(probe_smem) + (threadIdx.x & 31) * 8u;
    uint32_t q = (blockIdx.x * blockDim.x + threadIdx.x) * 977u, acc = 0;
    uint32_t a[4] = {q, q ^ 0x1234567u, q + 77u, q * 3u};
    float f[4] = {1.0f + (q & 7), 2.0f, 0.5f, 1.5f};
    constexpr int ILP = 4;
    for (int it = 0; it < iters; ++it) {
        uint32_t c0[ILP], c1[ILP], c2[ILP], c3[ILP];
#pragma unroll
        for (int j = 0; j < ILP; ++j) { c0[j] = q + j; c1[j] = sweep; c2[j] = slot; c3[j] = (uint32_t)it; }
        int ja = 0;
#pragma unroll
        for (int r = 0; r < 10; ++r) {
#pragma unroll
            for (int j = 0; j < ILP; ++j) {
                const uint32_t hi0 = __umulhi(kPhiloxM0, c0[j]), lo0 = kPhiloxM0 * c0[j];
                const uint32_t hi1 = __umulhi(kPhiloxM1, c2[j]), lo1 = kPhiloxM1 * c2[j];
                const uint32_t n0 = hi1 ^ c1[j] ^ rk.k[2 * r], n2 = hi0 ^ c3[j] ^ rk.k[2 * r + 1];
                c1[j] = lo1; c3[j] = lo0; c0[j] = n0; c2[j] = n2;
            }
#pragma unroll
            for (; ja < (r + 1) * N * ILP / 10; ++ja) probe_op<OP>(a, f, ja, saddr);
        }
        q += ILP;
#pragma unroll
        for (int j = 0; j < ILP; ++j) acc ^= c0[j] ^ c1[j] ^ c2[j] ^ c3[j];
    }
    acc ^= a[0] ^ a[1] ^ a[2] ^ a[3] ^ __float_as_uint(f[0] + f[1] + f[2] + f[3]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

__global__ void k_bench_stream(uint4* p, size_t n16) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) {
        uint4 q = p[i];
        q.x ^= 0x01010101u; q.y ^= 0x01010101u; q.z ^= 0x01010101u; q.w ^= 0x01010101u;
        p[i] = q;
    }
}

template <class F>
int time_launch(cudaStream_t s, F launch, double* ms) {
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return RFIM_ECUDA;
    launch();                                   // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(a, s);
        launch();
        cudaEventRecord(b, s);
        if (cudaEventSynchronize(b) != cudaSuccess) { cudaEventDestroy(a); cudaEventDestroy(b); return RFIM_ECUDA; }
        float t = 0.f;
        cudaEventElapsedTime(&t, a, b);
        best = std::min(best, t);
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    *ms = best;
    return cudaGetLastError() == cudaSuccess ? RFIM_OK : RFIM_ECUDA;
}

}  // namespace

extern "C" {

int rfim_pt_bench_philox(void* stream, int calls_per_thread, double* ms, double* attempts) {
    if (calls_per_thread < 1 || !ms || !attempts) return RFIM_EINVAL;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return RFIM_ECUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8, threads = 256;
    uint32_t* out = reinterpret_cast<uint32_t*>(dev_alloc((size_t)blocks * threads * 4));
    if (!out) return RFIM_ENOMEM;
    BenchKeys rk;
    {
        uint32_t k0 = 0x9E3779B9u, k1 = 0x1234567u;
        for (int r = 0; r < 10; ++r) { rk.k[2 * r] = k0; rk.k[2 * r + 1] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
    }
    const int calls = (calls_per_thread + 3) / 4 * 4;
    int rc = time_launch(s, [&] { k_bench_philox<<<blocks, threads, 0, s>>>(out, calls, rk, 7u, 3u); }, ms);
    dev_free(out);
    *attempts = 4.0 * (double)blocks * threads * calls;
    return rc;
}

int rfim_pt_bench_issue(void* stream, int kind, int extra_per_call, double* ms, double* warp_rows) {
    if (kind < 0 || kind >= kProbeKinds || (extra_per_call != 0 && extra_per_call != 8) || !ms || !warp_rows) return RFIM_EINVAL;
    if ((kind == kProbeNone) != (extra_per_call == 0)) return RFIM_EINVAL;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return RFIM_ECUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms, threads = 512, iters = 2000;             // one CTA of 16 warps per SM, like the sweep kernel
    const size_t smem = 200 * 1024;
    uint32_t* out = reinterpret_cast<uint32_t*>(dev_alloc((size_t)blocks * threads * 4));
    if (!out) return RFIM_ENOMEM;
    BenchKeys rk;
    {
        uint32_t k0 = 0x9E3779B9u, k1 = 0x1234567u;
        for (int r = 0; r < 10; ++r) { rk.k[2 * r] = k0; rk.k[2 * r + 1] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
    }
    int rc = RFIM_EINVAL;
#define RFIM_PROBE_CASE(K)                                                                                              \
    case K: {                                                                                                            \
        auto kern = k_bench_issue<K, (K == kProbeNone ? 0 : 8)>;                                                          \
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { rc = RFIM_ECUDA; break; } \
        rc = time_launch(s, [&] { kern<<<blocks, threads, smem, s>>>(out, iters, rk, 7u, 3u); }, ms);                     \
        break;                                                                                                            \
    }
    switch (kind) {
        RFIM_PROBE_CASE(kProbeNone) RFIM_PROBE_CASE(kProbeLop3) RFIM_PROBE_CASE(kProbePrmt) RFIM_PROBE_CASE(kProbeI2fp) RFIM_PROBE_CASE(kProbeI2fRm)
        RFIM_PROBE_CASE(kProbeFfma) RFIM_PROBE_CASE(kProbeFadd) RFIM_PROBE_CASE(kProbeMufu) RFIM_PROBE_CASE(kProbeLds64)
        default: break;
    }
#undef RFIM_PROBE_CASE
    dev_free(out);
    *warp_rows = (double)iters * 4 /* calls */ * 4 /* attempts per call */ * (threads / 32 / 4);   // per SM sub-partition
    return rc;
}

int rfim_pt_bench_stream(void* stream, size_t bytes, double* ms, double* bytes_moved) {
    if (bytes < 16 || !ms || !bytes_moved) return RFIM_EINVAL;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return RFIM_ECUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    uint4* p = reinterpret_cast<uint4*>(dev_alloc(bytes));
    if (!p) return RFIM_ENOMEM;
    cudaMemsetAsync(p, 0, bytes, s);
    const size_t n16 = bytes / 16;
    int rc = time_launch(s, [&] { k_bench_stream<<<sms * 8, 512, 0, s>>>(p, n16); }, ms);
    dev_free(p);
    *bytes_moved = 2.0 * (double)n16 * 16.0;
    return rc;
}

}  // extern "C"

// ---- an entry point that allocates nothing (include/rfim_pt.h: rfim_pt_energy_terms_noalloc) ----------------------
// For callers that may not call cudaMalloc (CUDA graph capture, tight serving loops): the energy / magnetisation
// reduction of k_reduce_site (S5; Eq. 1) over caller-owned DEVICE arrays in the boundary's
// natural site order, with its scratch (per-CTA partial sums and one arrival counter per replica) in a file-scope
// device array instead of a handle's cudaMalloc'ed accumulators.  Every GPU that loads the library holds the array until
// exit.  In host code `g_noalloc_scratch` is a host-side stand-in, NOT a device address: the launch code below takes the
// device address from cudaGetSymbolAddress, once per device, and passes that to the kernel.
namespace {

constexpr int kNoAllocMaxR = RFIM_PT_NOALLOC_MAX_R;      // replicas per call
constexpr int kNoAllocMaxL = RFIM_PT_NOALLOC_MAX_L;      // lattice side per call
constexpr int kNoAllocParts = 16;                        // CTAs (partial sums) per replica
constexpr int kNoAllocThreads = 256;
constexpr size_t kNoAllocPartWords = (size_t)kNoAllocMaxR * kNoAllocParts * 3;   // long long [R][part][Eb, Ef, Msum]
constexpr size_t kNoAllocWords = kNoAllocPartWords + kNoAllocMaxR / 2;           // + uint32 arrival counters [R]
constexpr int kNoAllocMaxDevices = 64;

static __device__ __align__(256) long long g_noalloc_scratch[kNoAllocWords];     // 98 304 + 1 024 bytes
static_assert(sizeof(long long) * kNoAllocWords == RFIM_PT_NOALLOC_SCRATCH_BYTES, "rfim_pt.h states the scratch size");

// grid (kNoAllocParts, R).  Eb = sum_i s_i (s_{i+x} + s_{i+y} + s_{i+z}) with periodic wrap counts every bond of
// k_reduce_site's colour-0 six-neighbour sum once (L = 2: twice, as there).  Pass 1: each CTA's partial sums go to
// scratch; pass 2: the last CTA of a replica to arrive adds them in CTA order, writes terms[r][3] and re-arms the counter.
__global__ void k_energy_terms_noalloc(int L, int kind, const int8_t* __restrict__ spins, const int32_t* __restrict__ field,
                                       long long* __restrict__ terms, long long* scratch) {
    const int r = blockIdx.y, parts = gridDim.x;
    const long long N = (long long)L * L * L;
    const int8_t* s = spins + (long long)r * N;
    long long* part = scratch + ((long long)r * kNoAllocParts + blockIdx.x) * 3;
    unsigned int* arrived = reinterpret_cast<unsigned int*>(scratch + kNoAllocPartWords) + r;
    long long eb = 0, ef = 0, ms = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)parts * blockDim.x) {
        const int x = (int)(i % L), y = (int)((i / L) % L), z = (int)(i / ((long long)L * L));
        const long long ix = i + (x + 1 == L ? 1 - L : 1);
        const long long iy = i + (long long)L * (y + 1 == L ? 1 - L : 1);
        const long long iz = i + (long long)L * L * (z + 1 == L ? 1 - L : 1);
        const int si = s[i];
        eb += si * ((int)s[ix] + (int)s[iy] + (int)s[iz]);
        ms += si;
        ef += kind == 0 ? (long long)(field[i] > 0 ? si : -si) : (long long)si * field[i];
    }
    __shared__ long long red[3][kNoAllocThreads / 32];
    __shared__ bool last;
    eb = warp_sum(eb); ef = warp_sum(ef); ms = warp_sum(ms);
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = eb; red[1][threadIdx.x >> 5] = ef; red[2][threadIdx.x >> 5] = ms; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 0; q < 3; ++q) {
            long long a = 0;
            for (int w = 0; w < kNoAllocThreads / 32; ++w) a += red[q][w];
            __stcg(part + q, a);
        }
        __threadfence();                                         // partial sums visible before the arrival is
        last = atomicAdd(arrived, 1u) == (unsigned int)parts - 1;
    }
    __syncthreads();
    if (!last) return;
    if (threadIdx.x < 3) {
        __threadfence();
        long long a = 0;
        for (int p = 0; p < parts; ++p) a += __ldcg(scratch + ((long long)r * kNoAllocParts + p) * 3 + threadIdx.x);
        terms[(long long)r * 3 + threadIdx.x] = a;
    }
    if (threadIdx.x == 0) *arrived = 0;                          // the next call on this stream finds it at zero
}

thread_local char g_noalloc_err[256] = "";

int noalloc_fail(int code, const char* what, const char* detail = "") {
    std::snprintf(g_noalloc_err, sizeof g_noalloc_err, "%s%s", what, detail);
    return code;
}

// device address of g_noalloc_scratch on the current device, looked up once per device
int noalloc_scratch(long long** out) {
    static long long* ptr[kNoAllocMaxDevices] = {};
    static std::mutex mu;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return noalloc_fail(RFIM_ECUDA, "cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return noalloc_fail(RFIM_EINVAL, "device ordinal beyond the scratch table");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        long long* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) return noalloc_fail(RFIM_ECUDA, "cudaGetSymbolAddress(g_noalloc_scratch): ", cudaGetErrorString(e));
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return RFIM_OK;
}

}  // namespace

extern "C" {

int rfim_pt_energy_terms_noalloc(void* cuda_stream, int L, int R, int field_kind, const int8_t* spins_device,
                                 const int32_t* field_device, int64_t* terms_device) {
    char lim[160];
    if (L < 2 || (L & 1)) return noalloc_fail(RFIM_EINVAL, "L must be even and >= 2");
    if (L > kNoAllocMaxL) {
        std::snprintf(lim, sizeof lim, "L = %d is beyond RFIM_PT_NOALLOC_MAX_L = %d", L, kNoAllocMaxL);
        return noalloc_fail(RFIM_EINVAL, lim);
    }
    if (R < 1) return noalloc_fail(RFIM_EINVAL, "R must be >= 1");
    if (R > kNoAllocMaxR) {
        std::snprintf(lim, sizeof lim, "R = %d is beyond RFIM_PT_NOALLOC_MAX_R = %d (the static scratch holds that many replicas)", R, kNoAllocMaxR);
        return noalloc_fail(RFIM_EINVAL, lim);
    }
    if (field_kind != RFIM_FIELD_BIMODAL && field_kind != RFIM_FIELD_GAUSSIAN) return noalloc_fail(RFIM_EINVAL, "bad field_kind");
    if (!spins_device || !field_device || !terms_device) return noalloc_fail(RFIM_EINVAL, "null device pointer");
    long long* scratch = nullptr;
    int rc = noalloc_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
    // the arrival counters must start at zero whatever an earlier (possibly failed) call left behind
    cudaError_t e = cudaMemsetAsync(scratch + kNoAllocPartWords, 0, sizeof(unsigned int) * kNoAllocMaxR, s);
    if (e != cudaSuccess) return noalloc_fail(RFIM_ECUDA, "cudaMemsetAsync: ", cudaGetErrorString(e));
    k_energy_terms_noalloc<<<dim3(kNoAllocParts, R), kNoAllocThreads, 0, s>>>(L, field_kind, spins_device, field_device,
                                                                             reinterpret_cast<long long*>(terms_device), scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc_fail(RFIM_ECUDA, "k_energy_terms_noalloc launch: ", cudaGetErrorString(e));
    g_noalloc_err[0] = 0;
    return RFIM_OK;
}

const char* rfim_pt_noalloc_last_error(void) { return g_noalloc_err; }

}  // extern "C"

#ifdef RFIM_RES_TIMING
extern "C" int rfim_pt_debug_timing(unsigned long long* out /* [256][8] */) {
    return cudaMemcpyFromSymbol(out, rfim::g_res_timing, sizeof(unsigned long long) * 256 * 8) == cudaSuccess ? 0 : -1;
}
#endif
