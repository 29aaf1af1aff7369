// rbg.cu -- host side of librbg.so: the C ABI of include/rbg.h over the kernels in rbg_kernels.cuh.
//
// Validation, role expansion (Eq. 19), role constants, launch
// geometry.  No CPU fallback: every step of the path runs in the CUDA kernels; this file only
// marshals.  Shares no code with oracle/.
#include "../../include/rbg.h"

#include <array>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <set>
#include <type_traits>
#include <utility>
#include <string>
#include <vector>

#include "rbg_kernels.cuh"
#include "rbg_be_kernels.cuh"

namespace {

thread_local std::string g_create_error;

struct Role {
    int process;           // index of the process the role comes from
    double sym_override;   // the process's sym field (< 0: paper rule)
    int s[4];              // species of the grid particle 1, its partner 2 and the incident pair 3, 4
    int kind;
    double par[4];
    double sym;
    int index;             // global role index
    int sampler;           // RBG_SAMPLER_*
    double cl, cg;         // degrees-of-freedom factors of the loss and the gain direction (reading R21)
    bool elastic;          // s3 == s1 && s4 == s2
};

}  // namespace

struct rbg_handle {
    int nx = 0, ix_offset = 0;
    int nxyz[3] = {0, 0, 0};
    int n_species = 0;
    std::vector<rbg_species> species;
    std::vector<rbg_momentum_grid> grids;
    std::vector<size_t> np, sp_off;
    std::vector<Role> roles;
    size_t f_elems = 0;
    double hbar = 1.0;
    int flags = 0;
    int device = 0;
    int sm_count = 148;
    int max_smem_optin = 0;
    // options
    int opt_warps = 0, opt_p1_per_cta = 0, opt_gather = 0, opt_spl = 0, opt_moments_path = 0, opt_vlasov_path = 0, opt_sym_tables = 0;
    int last_launches = 0;
    std::map<std::array<int, 4>, int> tile_cache;      // tile size chosen by run_roles per (role, cells, n_samples, warps)
    // per-species device tables for the moment / drift / Vlasov kernels: 1/E_p and v = p/E_p per momentum cell
    std::vector<double*> tab_iE, tab_v;
    double* charges_dev = nullptr;
    double2* dir_tab = nullptr;          // direction table of the double chain (rbg::kDirTabEntries entries)
    // scratch for the host entry point
    double *scratch_f = nullptr, *scratch_c = nullptr;
    int* scratch_flag = nullptr;         // negative-cell counter of rbg_collision_update_host
    size_t scratch_elems = 0;
    enum { HOST_CHUNKS_MAX = 16 };
    cudaStream_t host_streams[3] = {nullptr, nullptr, nullptr};      // copy-in, kernels, copy-out of rbg_collision_host
    cudaEvent_t host_events[2 * HOST_CHUNKS_MAX] = {};
    mutable std::string err;
};

namespace {

int fail(rbg_handle* h, int code, const std::string& msg) {
    if (h) h->err = msg; else g_create_error = msg;
    return code;
}

// Do the byte ranges [a, a + na) and [b, b + nb) share a byte?  Every kernel here reads f at cells other than the one it
// writes (gathers, stencil neighbours), so an output that overlaps the input even partly would be read half-updated.
bool ranges_overlap(const void* a, size_t na, const void* b, size_t nb) {
    const uintptr_t pa = reinterpret_cast<uintptr_t>(a), pb = reinterpret_cast<uintptr_t>(b);
    return pa < pb + nb && pb < pa + na;
}

// Makes the handle's device current for the duration of an entry point and restores the caller's on every exit path.
struct DeviceGuard {
    int prev = -1; int want;
    explicit DeviceGuard(int w) : want(w) { cudaGetDevice(&prev); if (prev != want) cudaSetDevice(want); }
    ~DeviceGuard() { if (prev >= 0 && prev != want) cudaSetDevice(prev); }
};

#define RBG_CUDA(h, call)                                                                          \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(h, RBG_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));        \
    } while (0)

// Role constants: the formulas of DESIGN.md section 4 ("role constants"), evaluated in double and then
// rounded to R.
template <typename R>
rbg::RoleParams<R> make_role_params(const rbg_handle& H, const Role& r) {
    rbg::RoleParams<R> k;
    std::memset(&k, 0, sizeof k);
    // masses of the four slots and their squares (each square rounded once, as DESIGN.md section 4 states the constants)
    double m[4], q[4];
    for (int i = 0; i < 4; ++i) { m[i] = H.species[r.s[i]].mass; q[i] = m[i] * m[i]; }
    k.m1 = (R)m[0]; k.m2 = (R)m[1];
    k.msq1 = (R)q[0]; k.msq2 = (R)q[1];
    k.m1m2 = (R)(m[0] * m[1]);
    // thresholds: (m1 + m2)^2, and its distance to (m3 + m4)^2 (0 for an elastic role); (m3 - m4)^2 and m3^2 - m4^2
    const double in_pair = m[0] + m[1], out_pair = m[2] + m[3], out_split = m[2] - m[3];
    const double in_pair2 = in_pair * in_pair;
    k.msum2 = (R)in_pair2;
    k.Mth = (R)(in_pair2 - out_pair * out_pair);
    k.Mdf = (R)(out_split * out_split);
    k.dm34 = (R)(q[2] - q[3]);
    k.msqsum = (R)((q[0] + q[1]) + (q[2] + q[3]));
    const rbg_momentum_grid& g1 = H.grids[r.s[0]];
    const rbg_momentum_grid& g2 = H.grids[r.s[1]];
    const rbg_momentum_grid& g3 = H.grids[r.s[2]];
    const rbg_momentum_grid& g4 = H.grids[r.s[3]];
    for (int d = 0; d < 3; ++d) {
        const double L1 = g1.pmax[d] - g1.pmin[d], L2 = g2.pmax[d] - g2.pmin[d];
        const double invD3 = (double)g3.n[d] / (g3.pmax[d] - g3.pmin[d]), invD4 = (double)g4.n[d] / (g4.pmax[d] - g4.pmin[d]);
        k.pmin1[d] = (R)g1.pmin[d];
        k.delta1[d] = (R)(L1 / (double)g1.n[d]);
        k.pmin2[d] = (R)g2.pmin[d];
        k.L2[d] = (R)L2;
        k.invD3[d] = (R)invD3; k.off3[d] = (R)(-g3.pmin[d] * invD3);
        k.invD4[d] = (R)invD4; k.off4[d] = (R)(-g4.pmin[d] * invD4);
        k.n1[d] = g1.n[d]; k.n2[d] = g2.n[d]; k.n3[d] = g3.n[d]; k.n4[d] = g4.n[d];
    }
    const double V2 = (g2.pmax[0] - g2.pmin[0]) * (g2.pmax[1] - g2.pmin[1]) * (g2.pmax[2] - g2.pmin[2]);
    const double tph = 2.0 * M_PI * H.hbar;
    R* tk[4] = {&k.tk1, &k.tk2, &k.tk3, &k.tk4};
    for (int i = 0; i < 4; ++i) *tk[i] = (R)((double)H.species[r.s[i]].stat * (tph * tph * tph) / H.species[r.s[i]].g);
    k.par0 = (R)(r.kind == RBG_M2_ISO_DSIGMA ? 64.0 * M_PI * M_PI * r.par[0] : r.par[0]);
    k.mD2 = (R)(r.par[1] * r.par[1]);
    k.twomD2 = (R)(2.0 * (r.par[1] * r.par[1]));
    const double g2c = r.par[0] * r.par[0];
    k.g4 = (R)(g2c * g2c);
    // Table III prefactors: the colour factors of SU(N_c = 3) (PAPER.md:671 quotes d_F = C_A = 3, C_F = 4/3, d_A = 8; here
    // from N_c: d_F = C_A = N_c, d_A = N_c^2 - 1, C_F = d_A / (2 N_c)), each times g^4 = par0^4 at the end
    const double Nc = 3.0, dF = Nc, CA = Nc, dA = Nc * Nc - 1.0, CF = dA / (2.0 * Nc);
    const double g4d = g2c * g2c, dFCF = dF * CF;
    k.qA = (R)(g4d * (8.0 * dFCF * dFCF / dA));
    k.qB = (R)(g4d * (16.0 * dFCF * (CF - 0.5 * CA)));
    k.qC = (R)(g4d * (8.0 * dFCF * CF));
    k.qD = (R)(g4d * (8.0 * dFCF * CA));
    k.qG = (R)(g4d * (16.0 * dA * (CA * CA)));
    k.qcd = r.kind >= RBG_M2_QCD_Q1Q2 ? r.kind - RBG_M2_QCD_Q1Q2 : 0;
    k.rho = (R)(r.cg / r.cl);
    k.symV2 = (H.hbar * H.hbar) * (r.sym * V2) * r.cl;     // hbar^2 c of Eq. 16, c = 1
    for (int i = 0; i < 4; ++i) k.np[i] = (int)H.np[r.s[i]];
    k.role = r.index;
    return k;
}

// Opt a kernel in to the device's largest dynamic shared-memory size once per (kernel, device) instead of before every
// launch.  Keyed by the kernel's address: kernels of one signature share a function-pointer type.
template <typename K>
cudaError_t ensure_max_smem(K kern, int device, int max_optin) {
    static std::mutex mu;
    static std::set<std::pair<const void*, int>> done;
    const std::pair<const void*, int> key(reinterpret_cast<const void*>(kern), device);
    std::lock_guard<std::mutex> lock(mu);
    if (done.count(key)) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, max_optin);
    if (e == cudaSuccess) done.insert(key);
    return e;
}
struct LaunchCtx { int device, max_optin; cudaStream_t st; };

template <typename R, int KIND, bool Q, bool SMEM, int MAXT, int SPL, bool TCH, bool INEL>
cudaError_t launch_one(const rbg::RoleParams<R>& rp, const rbg::LaunchParams& lp, int grid, int threads, size_t smem,
                       const LaunchCtx& cx) {
    auto kern = rbg::collision_role_kernel<R, KIND, Q, SMEM, MAXT, SPL, TCH, INEL>;
    const cudaError_t e = ensure_max_smem(kern, cx.device, cx.max_optin);
    if (e != cudaSuccess) return e;
    kern<<<grid, threads, smem, cx.st>>>(rp, lp);
    return cudaGetLastError();
}

// Launch geometries.  SPL = 2 samples per lane and loop iteration: the double chain in CTAs of up to 12 warps (384 threads,
// up to 168 registers per thread: 159 used, no spills, no constant re-loads in the loop), the float chain in CTAs of up to
// 16 warps (128 registers).  Wider CTAs (up to 32 warps, 64 registers) evaluate SPL = 1 (elastic roles only).  Results are
// bit-identical (fixed lane summation order).  Measured on config 4 / config 2 (profiles/r2_collision.md): 12 warps
// 9.66e10 / 9.18e10 samples/s, 16 warps at 128 registers 9.33e10 / 8.88e10, 8 / 10 / 11 / 13 warps 8.98 / 8.10 / 8.85 /
// 7.54e10 (warp counts that do not divide over the four schedulers lose); 4 samples per lane at 8 warps is 2-5 % slower
// than SPL = 2; the float chain gains nothing from 20-24 warps.
// (Table III kinds, row as a compile-time constant inside the kernel: config 7 runs 7.65e10 samples/s with 12 warps at 160
// registers, 7.50e10 with 16 at 128; with the row as a run-time switch in the sample loop it was 7.2e10 / 6.7e10)
template <typename R, int KIND> constexpr int kSpl2Threads = sizeof(R) == 8 ? 384 : 512;
template <typename R, int KIND, bool Q, bool SMEM, bool TCH, bool INEL>
cudaError_t launch_geo(int spl, const rbg::RoleParams<R>& rp, const rbg::LaunchParams& lp, int grid, int threads,
                       size_t smem, const LaunchCtx& st) {
    if constexpr (!INEL)
        if (spl == 1) return launch_one<R, KIND, Q, SMEM, 1024, 1, TCH, INEL>(rp, lp, grid, threads, smem, st);
    return launch_one<R, KIND, Q, SMEM, kSpl2Threads<R, KIND>, 2, TCH, INEL>(rp, lp, grid, threads, smem, st);
}

// inel: general roles (species 3,4 differ from 1,2), uniform sampler only
template <typename R, int KIND, bool TCH>
cudaError_t launch_kq(bool q, bool smem_path, bool inel, int spl, const rbg::RoleParams<R>& rp, const rbg::LaunchParams& lp,
                      int grid, int threads, size_t smem, const LaunchCtx& st) {
    if (inel) {
        if (q) return smem_path ? launch_geo<R, KIND, true, true, false, true>(spl, rp, lp, grid, threads, smem, st)
                                : launch_geo<R, KIND, true, false, false, true>(spl, rp, lp, grid, threads, smem, st);
        return smem_path ? launch_geo<R, KIND, false, true, false, true>(spl, rp, lp, grid, threads, smem, st)
                         : launch_geo<R, KIND, false, false, false, true>(spl, rp, lp, grid, threads, smem, st);
    }
    if (q) return smem_path ? launch_geo<R, KIND, true, true, TCH, false>(spl, rp, lp, grid, threads, smem, st)
                            : launch_geo<R, KIND, true, false, TCH, false>(spl, rp, lp, grid, threads, smem, st);
    return smem_path ? launch_geo<R, KIND, false, true, TCH, false>(spl, rp, lp, grid, threads, smem, st)
                     : launch_geo<R, KIND, false, false, TCH, false>(spl, rp, lp, grid, threads, smem, st);
}

template <typename R>
int run_roles(rbg_handle* h, const double* f, double* out, bool update, double dt, int* neg_flag, int n_samples,
              uint64_t seed, cudaStream_t stream, int cell_begin = 0, int cell_count = -1) {
    // [cell_begin, cell_begin + cell_count) = the local spatial cells this call sweeps (default: all of them); the stream
    // key is the global cell index, so sweeping the cells in several calls gives the same result as one call
    const LaunchCtx st{h->device, h->max_smem_optin, stream};
    const int ncell = cell_count < 0 ? h->nx : cell_count;
    if (cell_begin == 0) h->last_launches = 0;
    // last role per species (update mode counts negatives there); species with no role: C = 0 / f_out = f
    std::vector<int> first_role(h->n_species, -1), last_role(h->n_species, -1);
    for (size_t i = 0; i < h->roles.size(); ++i) {
        if (first_role[h->roles[i].s[0]] < 0) first_role[h->roles[i].s[0]] = (int)i;
        last_role[h->roles[i].s[0]] = (int)i;
    }
    for (int s = 0; s < h->n_species; ++s) {
        if (first_role[s] >= 0) continue;
        const size_t n = (size_t)ncell * h->np[s], o = h->sp_off[s] + (size_t)cell_begin * h->np[s];
        if (update) {
            rbg::copy_count_kernel<<<h->sm_count * 4, 256, 0, stream>>>(f + o, out + o, n, neg_flag);
            RBG_CUDA(h, cudaGetLastError());
            ++h->last_launches;
        } else {
            RBG_CUDA(h, cudaMemsetAsync(out + o, 0, n * sizeof(double), stream));
        }
    }
    for (size_t ir = 0; ir < h->roles.size(); ++ir) {
        const Role& r = h->roles[ir];
        const rbg::RoleParams<R> rp = make_role_params<R>(*h, r);
        const bool inel = !r.elastic;
        // samples per lane: 2 (at most 12 / 16 warps, double / float chain) unless the option or a wider CTA asks for 1
        // (elastic roles only)
        const int np1 = rp.np[0];
        // widest CTA of the two-samples-per-lane kernels of this chain and kind
        const int kW2 = (r.kind >= RBG_M2_QCD_Q1Q2 ? kSpl2Threads<R, rbg::KIND_QCD> : kSpl2Threads<R, rbg::KIND_CONST>) / 32;
        int spl = h->opt_spl > 0 ? h->opt_spl : 2;
        int warps = h->opt_warps > 0 ? h->opt_warps : (spl == 2 ? kW2 : 32);
        if (inel && warps > kW2) warps = kW2;
        if (warps > kW2) spl = 1;
        if (inel) spl = 2;
        // Tile size T (momentum cells per CTA; one CTA per SM at a time): a CTA stages its tables (about 2 us + bytes at
        // 100 GB/s) and then takes ceil(T / warps) rounds of one p1 per warp (a round of n_samples samples per warp at
        // about 5.7e8 samples/s per SM); the grid of nx * tiles CTAs runs in ceil(nx * tiles / SMs) waves.  Take the
        // tiling with the smallest waves * (rounds + staging), preferring larger tiles on near-ties.  T <= 512.
        // The search takes up to 4096 candidates with several 64-bit divisions each, and its inputs never change inside a
        // time-step loop (rbg_collision_evolve), so its result is kept per (role, cells in the sweep, n_samples, warps).
        int T = h->opt_p1_per_cta;
        const std::array<int, 4> tile_key{(int)ir, ncell, n_samples, warps};
        const auto cached = T <= 0 ? h->tile_cache.find(tile_key) : h->tile_cache.end();
        if (cached != h->tile_cache.end()) T = cached->second;
        if (T <= 0) {
            size_t tab_bytes = 0;
            for (int i = 1; i < 4; ++i) {
                bool first = true;
                for (int j = 1; j < i; ++j) first = first && r.s[j] != r.s[i];
                if (first) tab_bytes += (size_t)rp.np[i] * sizeof(R);
            }
            const double staging = (2e-6 + (double)tab_bytes / 1e11) * 5.7e8 / ((double)n_samples * warps);
            double best_cost = -1.0;
            const int t_lo = (np1 + 511) / 512, t_hi = std::max(t_lo, std::min(4096, (np1 + warps - 1) / warps));
            for (int tiles = t_lo; tiles <= t_hi; ++tiles) {
                const int Tt = (np1 + tiles - 1) / tiles;
                const long ctas = (long)ncell * ((np1 + Tt - 1) / Tt);
                const double cost = (double)((ctas + h->sm_count - 1) / h->sm_count) * ((double)((Tt + warps - 1) / warps) + staging);
                if (best_cost < 0.0 || cost < 0.995 * best_cost) { best_cost = cost; T = Tt; }
            }
            h->tile_cache[tile_key] = T;
        }
        T = std::max(1, std::min(T, np1));
        // shared memory: [16 B mbarrier][T doubles][one f table per distinct species among slots 2, 3, 4, 16-B aligned]
        rbg::LaunchParams lp;
        std::memset(&lp, 0, sizeof lp);
        const size_t head = 16 + (sizeof(R) == 8 ? (size_t)rbg::kDirTabBytes : 0) + (((size_t)T * 8 + 15) & ~(size_t)15);
        size_t tabs = 0;
        for (int i = 1; i < 4; ++i) {
            int owner = i;
            for (int j = 1; j < i; ++j) if (r.s[j] == r.s[i]) { owner = j; break; }
            if (owner == i) {
                lp.tab_own[i] = 1; lp.tab_off[i] = (int)tabs;
                tabs += ((size_t)rp.np[i] * sizeof(R) + 15) & ~(size_t)15;
            } else {
                lp.tab_own[i] = 0; lp.tab_off[i] = lp.tab_off[owner];
            }
        }
        bool smem_path = head + tabs <= (size_t)h->max_smem_optin;
        if (h->opt_gather == 1 && !smem_path) return fail(h, RBG_E_UNSUPPORTED, "gather=1 (shared memory) requested but the f tables do not fit");
        if (h->opt_gather == 2) smem_path = false;
        const size_t smem = head + (smem_path ? tabs : 0);
        for (int i = 0; i < 4; ++i) lp.fb[i] = f + h->sp_off[r.s[i]] + (size_t)cell_begin * h->np[r.s[i]];
        lp.out_base = out + h->sp_off[r.s[0]] + (size_t)cell_begin * h->np[r.s[0]];
        lp.nx_local = ncell; lp.ix_offset = h->ix_offset + cell_begin; lp.n_samples = n_samples;
        lp.dir_tab = h->dir_tab;
        lp.key0 = (uint32_t)seed; lp.key1 = (uint32_t)(seed >> 32);
        for (int rr = 0; rr < 10; ++rr) {
            lp.rk[2 * rr] = lp.key0 + (uint32_t)rr * 0x9E3779B9u;
            lp.rk[2 * rr + 1] = lp.key1 + (uint32_t)rr * 0xBB67AE85u;
        }
        lp.p1_per_cta = T; lp.tiles = (np1 + T - 1) / T;
        lp.accumulate = first_role[r.s[0]] != (int)ir;
        lp.update = update; lp.dt = dt; lp.neg_flag = neg_flag;
        lp.count_negative = update && last_role[r.s[0]] == (int)ir;
        const long grid = (long)lp.tiles * ncell;
        if (grid > 0x7fffffffL) return fail(h, RBG_E_UNSUPPORTED, "grid too large; raise p1_per_cta");
        bool q = false;
        for (int i = 0; i < 4; ++i) q = q || h->species[r.s[i]].stat != 0;
        cudaError_t e;
        const bool tch = r.sampler == RBG_SAMPLER_TCHANNEL;
        const int th = warps * 32;
        switch (r.kind) {
            case RBG_M2_CONST: e = launch_kq<R, rbg::KIND_CONST, false>(q, smem_path, inel, spl, rp, lp, (int)grid, th, smem, st); break;
            case RBG_M2_COULOMB_SCREENED:
                e = tch ? launch_kq<R, rbg::KIND_COULOMB, true>(q, smem_path, inel, spl, rp, lp, (int)grid, th, smem, st)
                        : launch_kq<R, rbg::KIND_COULOMB, false>(q, smem_path, inel, spl, rp, lp, (int)grid, th, smem, st);
                break;
            case RBG_M2_TCHAN_S2:
                e = tch ? launch_kq<R, rbg::KIND_TCHAN_S2, true>(q, smem_path, inel, spl, rp, lp, (int)grid, th, smem, st)
                        : launch_kq<R, rbg::KIND_TCHAN_S2, false>(q, smem_path, inel, spl, rp, lp, (int)grid, th, smem, st);
                break;
            case RBG_M2_ISO_DSIGMA: e = launch_kq<R, rbg::KIND_ISO_DSIGMA, false>(q, smem_path, inel, spl, rp, lp, (int)grid, th, smem, st); break;
            default: e = launch_kq<R, rbg::KIND_QCD, false>(q, smem_path, inel, spl, rp, lp, (int)grid, th, smem, st); break;
        }
        if (e != cudaSuccess) return fail(h, RBG_E_CUDA, std::string("kernel launch: ") + cudaGetErrorString(e));
        ++h->last_launches;
    }
    return RBG_OK;
}

int run(rbg_handle* h, const double* f, double* out, bool update, double dt, int* neg_flag, int n_samples, uint64_t seed,
        void* stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f || !out) return fail(h, RBG_E_INVALID_ARG, "null buffer");
    if (ranges_overlap(f, h->f_elems * sizeof(double), out, h->f_elems * sizeof(double)))
        return fail(h, RBG_E_INVALID_ARG, "the output buffer overlaps f (the kernels gather f at other cells while they write)");
    if (n_samples <= 0) return fail(h, RBG_E_INVALID_ARG, "n_samples must be positive");
    if (update && !neg_flag) return fail(h, RBG_E_INVALID_ARG, "null neg_flag_dev");
    cudaStream_t st = (cudaStream_t)stream;
    DeviceGuard guard(h->device);
    return (h->flags & RBG_FP32_KINEMATICS) ? run_roles<float>(h, f, out, update, dt, neg_flag, n_samples, seed, st)
                                            : run_roles<double>(h, f, out, update, dt, neg_flag, n_samples, seed, st);
}

}  // namespace

namespace {
template <int KIND>
cudaError_t launch_sym(bool q, bool inel, bool csmem, const rbg::RoleParams<double>& rp, const rbg::LaunchParams& lp,
                       const rbg::SymParams& sp, int grid, size_t smem, const LaunchCtx& cx) {
    auto go = [&](auto kern) -> cudaError_t {
        const cudaError_t e = ensure_max_smem(kern, cx.device, cx.max_optin);
        if (e != cudaSuccess) return e;
        kern<<<grid, 512, smem, cx.st>>>(rp, lp, sp);
        return cudaGetLastError();
    };
    if (q) {
        if (inel) return csmem ? go(rbg::collision_symmetric_kernel<KIND, true, true, true>) : go(rbg::collision_symmetric_kernel<KIND, true, true, false>);
        return csmem ? go(rbg::collision_symmetric_kernel<KIND, true, false, true>) : go(rbg::collision_symmetric_kernel<KIND, true, false, false>);
    }
    if (inel) return csmem ? go(rbg::collision_symmetric_kernel<KIND, false, true, true>) : go(rbg::collision_symmetric_kernel<KIND, false, true, false>);
    return csmem ? go(rbg::collision_symmetric_kernel<KIND, false, false, true>) : go(rbg::collision_symmetric_kernel<KIND, false, false, false>);
}
}  // namespace

extern "C" {

int rbg_create(rbg_handle** out, const rbg_spatial_grid* grid, int n_species, const rbg_species* species,
               const rbg_momentum_grid* mg, int n_process, const rbg_process* processes, double hbar, int flags) {
    if (!out) return fail(nullptr, RBG_E_INVALID_ARG, "out is null");
    *out = nullptr;
    if (!grid || !species || !mg || (n_process > 0 && !processes)) return fail(nullptr, RBG_E_INVALID_ARG, "null argument");
    if (grid->nx <= 0 || grid->ny <= 0 || grid->nz <= 0 || grid->ix_offset < 0)
        return fail(nullptr, RBG_E_INVALID_ARG, "spatial grid counts must be positive");
    if ((long)grid->nx * grid->ny * grid->nz > 0x7fffffffL) return fail(nullptr, RBG_E_INVALID_ARG, "too many spatial cells");
    if (n_species <= 0 || n_process < 0) return fail(nullptr, RBG_E_INVALID_ARG, "bad species/process count");
    if (!(hbar > 0.0)) return fail(nullptr, RBG_E_INVALID_ARG, "hbar must be positive");
    if (flags != RBG_FP64 && flags != RBG_FP32_KINEMATICS) return fail(nullptr, RBG_E_INVALID_ARG, "unknown flags");
    rbg_handle* h = new rbg_handle;
    h->nx = grid->nx * grid->ny * grid->nz;
    h->nxyz[0] = grid->nx; h->nxyz[1] = grid->ny; h->nxyz[2] = grid->nz;
    h->ix_offset = grid->ix_offset;
    h->n_species = n_species; h->hbar = hbar; h->flags = flags;
    size_t off = 0;
    for (int s = 0; s < n_species; ++s) {
        const rbg_species& S = species[s];
        const rbg_momentum_grid& G = mg[s];
        std::string why;
        if (!(S.mass >= 0.0)) why = "negative mass";
        else if (S.stat != 0 && S.stat != 1 && S.stat != -1) why = "stat must be 0, +1 or -1";
        else if (!(S.g > 0.0)) why = "g must be positive";
        for (int d = 0; d < 3 && why.empty(); ++d) {
            if (G.n[d] <= 0) why = "momentum grid counts must be positive";
            else if (!(G.pmax[d] > G.pmin[d])) why = "pmax must exceed pmin";
        }
        const double npd = (double)G.n[0] * G.n[1] * G.n[2];
        if (why.empty() && npd > 0x7fffffff) why = "too many momentum cells";
        if (!why.empty()) { delete h; return fail(nullptr, RBG_E_INVALID_ARG, "species " + std::to_string(s) + ": " + why); }
        h->species.push_back(S); h->grids.push_back(G);
        h->np.push_back((size_t)npd); h->sp_off.push_back(off);
        off += (size_t)h->nx * (size_t)npd;
    }
    h->f_elems = off;
    for (int i = 0; i < n_process; ++i) {
        const rbg_process& p = processes[i];
        const int idx[4] = {p.a, p.b, p.c, p.d};
        for (int j = 0; j < 4; ++j)
            if (idx[j] < 0 || idx[j] >= n_species) { delete h; return fail(nullptr, RBG_E_INVALID_ARG, "process " + std::to_string(i) + ": species index out of range"); }
        // 1/p^0 of Eq. 16: a species that takes part in a process must have no momentum cell whose centre
        // has (numerically) zero energy -- a massless species on an odd grid symmetric about 0 (reading R14)
        for (int j = 0; j < 4; ++j) {
            const rbg_momentum_grid& G = mg[idx[j]];
            double e2 = species[idx[j]].mass * species[idx[j]].mass, wmin = 0.0;
            for (int d = 0; d < 3; ++d) {
                const double w = (G.pmax[d] - G.pmin[d]) / (double)G.n[d];
                // centre nearest to 0 along this axis: cell floor(-pmin / w) or one of its neighbours
                const double c0 = std::floor(-G.pmin[d] / w);
                double best = HUGE_VAL;
                for (double c = c0 - 1.0; c <= c0 + 1.0; c += 1.0) {
                    if (c < 0.0 || c > (double)(G.n[d] - 1)) continue;
                    best = std::fmin(best, std::fabs(std::fma(c + 0.5, w, G.pmin[d])));
                }
                if (best == HUGE_VAL) best = std::fmin(std::fabs(std::fma(0.5, w, G.pmin[d])), std::fabs(std::fma((double)G.n[d] - 0.5, w, G.pmin[d])));
                e2 += best * best;
                wmin = d == 0 ? w : std::fmin(wmin, w);
            }
            if (!(std::sqrt(e2) > 1e-6 * wmin)) {
                delete h;
                return fail(nullptr, RBG_E_UNSUPPORTED, "process " + std::to_string(i) + ": species " + std::to_string(idx[j]) +
                            " has a momentum cell centre with zero energy (massless, centre at p = 0): 1/p0 of Eq. 16 diverges there");
            }
        }
        if (p.kind < RBG_M2_CONST || p.kind > RBG_M2_QCD_GG) { delete h; return fail(nullptr, RBG_E_INVALID_ARG, "process " + std::to_string(i) + ": unknown |M|^2 kind"); }
        const bool elastic = p.c == p.a && p.d == p.b;
        if (!elastic && p.c == p.b && p.d == p.a) { delete h; return fail(nullptr, RBG_E_INVALID_ARG, "process " + std::to_string(i) + ": write a+b -> b+a as a+b -> a+b (t and u would be ambiguous)"); }
        if (p.sampler != RBG_SAMPLER_UNIFORM && p.sampler != RBG_SAMPLER_TCHANNEL) { delete h; return fail(nullptr, RBG_E_INVALID_ARG, "process " + std::to_string(i) + ": unknown sampler"); }
        if (p.sampler == RBG_SAMPLER_TCHANNEL && !(elastic && (p.kind == RBG_M2_COULOMB_SCREENED || p.kind == RBG_M2_TCHAN_S2) && p.par[1] != 0.0)) {
            delete h;
            return fail(nullptr, RBG_E_INVALID_ARG, "process " + std::to_string(i) + ": the t-channel sampler needs an elastic process of a t-channel |M|^2 kind with a non-zero regulator par[1]");
        }
        // Role expansion: a+b -> c+d seen from a, from b, and, if inelastic, from c and from d.
        // DOF factors (reading R21): Table III kinds are summed over the DOF of all four particles; kinds 0..3 are
        // averaged over those of a and b.
        const double sum_norm = p.kind >= RBG_M2_QCD_Q1Q2 ? 1.0 : species[p.a].g * species[p.b].g;
        Role r;
        r.process = i; r.sym_override = p.sym;
        r.sampler = p.sampler;
        r.kind = p.kind; std::memcpy(r.par, p.par, sizeof r.par);
        r.elastic = elastic;
        auto add = [&](int s1, int s2, int s3, int s4) {
            r.s[0] = s1; r.s[1] = s2; r.s[2] = s3; r.s[3] = s4;
            r.sym = p.sym < 0 ? (s3 == s4 ? 0.5 : 1.0) : p.sym;
            r.cl = sum_norm / (species[s1].g * species[s2].g);
            r.cg = sum_norm / (species[s3].g * species[s4].g);
            r.index = (int)h->roles.size();
            h->roles.push_back(r);
        };
        add(p.a, p.b, p.c, p.d);
        if (p.b != p.a) add(p.b, p.a, p.d, p.c);
        if (!elastic) {
            add(p.c, p.d, p.a, p.b);
            if (p.d != p.c) add(p.d, p.c, p.b, p.a);
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { delete h; return fail(nullptr, RBG_E_CUDA, "no CUDA device (there is no CPU fallback)"); }
    cudaGetDevice(&h->device);
    cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, h->device);
    cudaDeviceGetAttribute(&h->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    // momentum-cell tables (E_p = sqrt(|p|^2 + m^2); v = p / E_p, Eq. 6): inputs of the NEXT-4 kernels
    std::vector<double> charges(n_species);
    for (int s = 0; s < n_species; ++s) {
        const rbg_momentum_grid& G = h->grids[s];
        const size_t np = h->np[s];
        std::vector<double> iE(np), v(3 * np);
        const double m = h->species[s].mass;
        charges[s] = h->species[s].charge;
        size_t j = 0;
        for (int i0 = 0; i0 < G.n[0]; ++i0)
            for (int i1 = 0; i1 < G.n[1]; ++i1)
                for (int i2 = 0; i2 < G.n[2]; ++i2, ++j) {
                    const int id[3] = {i0, i1, i2};
                    double pc[3];
                    for (int d = 0; d < 3; ++d) pc[d] = G.pmin[d] + ((double)id[d] + 0.5) * ((G.pmax[d] - G.pmin[d]) / (double)G.n[d]);
                    const double E = std::sqrt(((pc[0] * pc[0] + pc[1] * pc[1]) + pc[2] * pc[2]) + m * m);
                    iE[j] = E > 0.0 ? 1.0 / E : 0.0;
                    for (int d = 0; d < 3; ++d) v[(size_t)d * np + j] = E > 0.0 ? pc[d] / E : 0.0;
                }
        double *d_iE = nullptr, *d_v = nullptr;
        if (cudaMalloc(&d_iE, np * sizeof(double)) != cudaSuccess || cudaMalloc(&d_v, 3 * np * sizeof(double)) != cudaSuccess ||
            cudaMemcpy(d_iE, iE.data(), np * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(d_v, v.data(), 3 * np * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaFree(d_iE); cudaFree(d_v); rbg_destroy(h);
            return fail(nullptr, RBG_E_CUDA, "allocating the momentum-cell tables failed");
        }
        h->tab_iE.push_back(d_iE); h->tab_v.push_back(d_v);
    }
    // direction table of the double chain (O6): evaluated once on the device
    if (cudaMalloc(&h->dir_tab, rbg::kDirTabBytes) != cudaSuccess) { rbg_destroy(h); return fail(nullptr, RBG_E_CUDA, "allocating the direction table failed"); }
    rbg::dir_table_kernel<<<(rbg::kDirTabEntries + 255) / 256, 256>>>(h->dir_tab);
    if (cudaGetLastError() != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) { rbg_destroy(h); return fail(nullptr, RBG_E_CUDA, "building the direction table failed"); }
    if (cudaMalloc(&h->charges_dev, n_species * sizeof(double)) != cudaSuccess ||
        cudaMemcpy(h->charges_dev, charges.data(), n_species * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess) {
        rbg_destroy(h);
        return fail(nullptr, RBG_E_CUDA, "allocating the charge table failed");
    }
    *out = h;
    return RBG_OK;
}

int rbg_collision(rbg_handle* h, const double* f_dev, double* C_dev, int n_samples, uint64_t seed, void* cuda_stream) {
    return run(h, f_dev, C_dev, false, 0.0, nullptr, n_samples, seed, cuda_stream);
}

int rbg_collision_update(rbg_handle* h, const double* f_dev, double* f_out_dev, double dt, int* neg_flag_dev,
                         int n_samples, uint64_t seed, void* cuda_stream) {
    return run(h, f_dev, f_out_dev, true, dt, neg_flag_dev, n_samples, seed, cuda_stream);
}

int rbg_collision_symmetric(rbg_handle* h, const double* f_dev, double* C_dev, int n_samples, uint64_t seed, void* cuda_stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f_dev || !C_dev) return fail(h, RBG_E_INVALID_ARG, "null buffer");
    if (ranges_overlap(f_dev, h->f_elems * sizeof(double), C_dev, h->f_elems * sizeof(double)))
        return fail(h, RBG_E_INVALID_ARG, "C_dev overlaps f_dev (the kernels gather f at other cells while they deposit)");
    if (n_samples <= 0) return fail(h, RBG_E_INVALID_ARG, "n_samples must be positive");
    if (h->flags & RBG_FP32_KINEMATICS) return fail(h, RBG_E_UNSUPPORTED, "rbg_collision_symmetric is fp64 only");
    for (const Role& r : h->roles)
        if (r.sampler != RBG_SAMPLER_UNIFORM) return fail(h, RBG_E_UNSUPPORTED, "rbg_collision_symmetric supports the uniform sampler only");
    DeviceGuard guard(h->device);
    const LaunchCtx st{h->device, h->max_smem_optin, (cudaStream_t)cuda_stream};
    h->last_launches = 0;
    RBG_CUDA(h, cudaMemsetAsync(C_dev, 0, h->f_elems * sizeof(double), st.st));
    auto dp3 = [&](int s) {
        const rbg_momentum_grid& g = h->grids[s];
        return ((g.pmax[0] - g.pmin[0]) / g.n[0]) * ((g.pmax[1] - g.pmin[1]) / g.n[1]) * ((g.pmax[2] - g.pmin[2]) / g.n[2]);
    };
    for (size_t ir = 0; ir < h->roles.size(); ++ir) {
        Role r = h->roles[ir];
        r.sym = 1.0;                                     // the symmetry factor is per slot here (SymParams::fac)
        const rbg::RoleParams<double> rp = make_role_params<double>(*h, r);
        rbg::SymParams sp;
        std::memset(&sp, 0, sizeof sp);
        for (int k = 0; k < 4; ++k) {
            int m = 0;                                   // (role, slot) pairs of the process that carry species s_k
            for (const Role& r2 : h->roles)
                if (r2.process == r.process)
                    for (int k2 = 0; k2 < 4; ++k2) m += r2.s[k2] == r.s[k];
            const int oa = k < 2 ? 2 : 0;                // the opposite pair
            const double symk = r.sym_override >= 0 ? r.sym_override : (r.s[oa] == r.s[oa + 1] ? 0.5 : 1.0);
            sp.fac[k] = (k < 2 ? 1.0 : -1.0) * symk * (dp3(r.s[0]) / dp3(r.s[k])) / (double)m;
            sp.cb[k] = C_dev + h->sp_off[r.s[k]];
        }
        // accumulator tables of the distinct species among slots 2..4
        size_t tabs = 0;
        for (int i = 1; i < 4; ++i) {
            int owner = i;
            for (int j = 1; j < i; ++j) if (r.s[j] == r.s[i]) { owner = j; break; }
            if (owner == i) { sp.ctab_own[i] = 1; sp.ctab_off[i] = (int)tabs; tabs += ((size_t)rp.np[i] * 8 + 15) & ~(size_t)15; }
            else { sp.ctab_own[i] = 0; sp.ctab_off[i] = sp.ctab_off[owner]; }
        }
        // Deposits go straight to C with red.global.add.f64 (one L2 atomic each) unless the option asks for per-CTA
        // shared-memory tables: sm_100 has no fp64 shared-memory atomic add (red.shared.add.f64 compiles to a compare-and-swap
        // loop), and the tables run 9-17 % slower (configs 4 / 7 / 2, profiles/r2_collision.md)
        const bool csmem = h->opt_sym_tables == 1 && rbg::kDirTabBytes + tabs <= (size_t)h->max_smem_optin;
        rbg::LaunchParams lp;
        std::memset(&lp, 0, sizeof lp);
        lp.dir_tab = h->dir_tab;
        for (int i = 0; i < 4; ++i) lp.fb[i] = f_dev + h->sp_off[r.s[i]];
        lp.nx_local = h->nx; lp.ix_offset = h->ix_offset; lp.n_samples = n_samples;
        lp.key0 = (uint32_t)seed; lp.key1 = (uint32_t)(seed >> 32);
        for (int rr = 0; rr < 10; ++rr) {
            lp.rk[2 * rr] = lp.key0 + (uint32_t)rr * 0x9E3779B9u;
            lp.rk[2 * rr + 1] = lp.key1 + (uint32_t)rr * 0xBB67AE85u;
        }
        // few, large tiles: every CTA flushes its tables with one global atomic per touched cell
        const int np1 = rp.np[0];
        int tiles = 1;
        while ((long)tiles * h->nx < 2L * h->sm_count && tiles * 32 < np1) tiles *= 2;
        lp.p1_per_cta = (np1 + tiles - 1) / tiles;
        lp.tiles = (np1 + lp.p1_per_cta - 1) / lp.p1_per_cta;
        const long grid = (long)lp.tiles * h->nx;
        if (grid > 0x7fffffffL) return fail(h, RBG_E_UNSUPPORTED, "grid too large");
        bool q = false;
        for (int i = 0; i < 4; ++i) q = q || h->species[r.s[i]].stat != 0;
        const size_t smem = rbg::kDirTabBytes + (csmem ? tabs : 0);
        cudaError_t e;
        switch (r.kind) {
            case RBG_M2_CONST: e = launch_sym<rbg::KIND_CONST>(q, !r.elastic, csmem, rp, lp, sp, (int)grid, smem, st); break;
            case RBG_M2_COULOMB_SCREENED: e = launch_sym<rbg::KIND_COULOMB>(q, !r.elastic, csmem, rp, lp, sp, (int)grid, smem, st); break;
            case RBG_M2_TCHAN_S2: e = launch_sym<rbg::KIND_TCHAN_S2>(q, !r.elastic, csmem, rp, lp, sp, (int)grid, smem, st); break;
            case RBG_M2_ISO_DSIGMA: e = launch_sym<rbg::KIND_ISO_DSIGMA>(q, !r.elastic, csmem, rp, lp, sp, (int)grid, smem, st); break;
            default: e = launch_sym<rbg::KIND_QCD>(q, !r.elastic, csmem, rp, lp, sp, (int)grid, smem, st); break;
        }
        if (e != cudaSuccess) return fail(h, RBG_E_CUDA, std::string("kernel launch: ") + cudaGetErrorString(e));
        ++h->last_launches;
    }
    return RBG_OK;
}

int rbg_collision_evolve(rbg_handle* h, double* f_dev, double* scratch_dev, double dt, int n_steps, int* neg_flag_dev,
                         int n_samples, uint64_t seed, void* cuda_stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (n_steps < 0) return fail(h, RBG_E_INVALID_ARG, "n_steps must be >= 0");
    if (!f_dev || !scratch_dev) return fail(h, RBG_E_INVALID_ARG, "null buffer");
    const size_t bytes = h->f_elems * sizeof(double);
    if (ranges_overlap(f_dev, bytes, scratch_dev, bytes)) return fail(h, RBG_E_INVALID_ARG, "scratch_dev overlaps f_dev");
    DeviceGuard guard(h->device);
    double *cur = f_dev, *nxt = scratch_dev;
    int launches = 0;
    for (int k = 0; k < n_steps; ++k) {
        const int rc = run(h, cur, nxt, true, dt, neg_flag_dev, n_samples, seed + (uint64_t)k, cuda_stream);
        if (rc != RBG_OK) return rc;
        launches += h->last_launches;
        std::swap(cur, nxt);
    }
    if (cur != f_dev) RBG_CUDA(h, cudaMemcpyAsync(f_dev, cur, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    h->last_launches = launches;
    return RBG_OK;
}

// Host-buffer sweep shared by rbg_collision_host (update = false: C into C_host) and rbg_collision_update_host (update =
// true: f + dt C into C_host, *neg_count_host = cells left negative).
static int host_sweep(rbg_handle* h, const double* f_host, double* C_host, bool update, double dt, int* neg_count_host,
                      int n_samples, uint64_t seed) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f_host || !C_host || (update && !neg_count_host)) return fail(h, RBG_E_INVALID_ARG, "null buffer");
    if (ranges_overlap(f_host, h->f_elems * sizeof(double), C_host, h->f_elems * sizeof(double)))
        return fail(h, RBG_E_INVALID_ARG, "C_host overlaps f_host (chunks of C are copied out while later chunks of f are still being read)");
    if (n_samples <= 0) return fail(h, RBG_E_INVALID_ARG, "n_samples must be positive");
    DeviceGuard guard(h->device);
    if (h->scratch_elems < h->f_elems) {
        cudaFree(h->scratch_f); cudaFree(h->scratch_c); h->scratch_f = h->scratch_c = nullptr; h->scratch_elems = 0;
        RBG_CUDA(h, cudaMalloc(&h->scratch_f, h->f_elems * sizeof(double)));
        RBG_CUDA(h, cudaMalloc(&h->scratch_c, h->f_elems * sizeof(double)));
        h->scratch_elems = h->f_elems;
    }
    if (update && !h->scratch_flag) RBG_CUDA(h, cudaMalloc(&h->scratch_flag, sizeof(int)));
    if (!h->host_streams[0]) {
        for (int i = 0; i < 3; ++i) RBG_CUDA(h, cudaStreamCreateWithFlags(&h->host_streams[i], cudaStreamNonBlocking));
        for (int i = 0; i < 2 * rbg_handle::HOST_CHUNKS_MAX; ++i) RBG_CUDA(h, cudaEventCreateWithFlags(&h->host_events[i], cudaEventDisableTiming));
    }
    // Spatial cells are independent (Eq. 16 couples only momenta at one x), so the sweep is pipelined over chunks of cells:
    // copy-in of chunk k+1 and copy-out of chunk k-1 run beside the kernels of chunk k (three streams).  The chunk count
    // keeps a chunk at 64 MB or more; small problems take one chunk.  Results do not depend on it (global-cell stream key).
    const size_t bytes = h->f_elems * sizeof(double);
    int chunks = (int)std::min<size_t>(rbg_handle::HOST_CHUNKS_MAX, std::max<size_t>(1, bytes / ((size_t)64 << 20)));
    chunks = std::min(chunks, h->nx);
    cudaStream_t s_in = h->host_streams[0], s_k = h->host_streams[1], s_out = h->host_streams[2];
    const bool fp32 = (h->flags & RBG_FP32_KINEMATICS) != 0;
    // The pipeline queues copies into and out of the CALLER's host buffers on three streams.  Whatever happens, this call
    // returns only after all three have drained: after an error return the caller may free or reuse f_host / C_host at
    // once, and no DMA may still be running on them then.
    int neg_count = 0;
    auto pipeline = [&]() -> int {
        if (update) RBG_CUDA(h, cudaMemsetAsync(h->scratch_flag, 0, sizeof(int), s_k));
        for (int c = 0; c < chunks; ++c) {
            const int x0 = (int)((long)h->nx * c / chunks), x1 = (int)((long)h->nx * (c + 1) / chunks);
            for (int s = 0; s < h->n_species; ++s) {
                const size_t o = h->sp_off[s] + (size_t)x0 * h->np[s], n = (size_t)(x1 - x0) * h->np[s];
                RBG_CUDA(h, cudaMemcpyAsync(h->scratch_f + o, f_host + o, n * sizeof(double), cudaMemcpyHostToDevice, s_in));
            }
            RBG_CUDA(h, cudaEventRecord(h->host_events[2 * c], s_in));
            RBG_CUDA(h, cudaStreamWaitEvent(s_k, h->host_events[2 * c], 0));
            const int rc = fp32 ? run_roles<float>(h, h->scratch_f, h->scratch_c, update, dt, h->scratch_flag, n_samples, seed, s_k, x0, x1 - x0)
                                : run_roles<double>(h, h->scratch_f, h->scratch_c, update, dt, h->scratch_flag, n_samples, seed, s_k, x0, x1 - x0);
            if (rc != RBG_OK) return rc;
            RBG_CUDA(h, cudaEventRecord(h->host_events[2 * c + 1], s_k));
            RBG_CUDA(h, cudaStreamWaitEvent(s_out, h->host_events[2 * c + 1], 0));
            for (int s = 0; s < h->n_species; ++s) {
                const size_t o = h->sp_off[s] + (size_t)x0 * h->np[s], n = (size_t)(x1 - x0) * h->np[s];
                RBG_CUDA(h, cudaMemcpyAsync(C_host + o, h->scratch_c + o, n * sizeof(double), cudaMemcpyDeviceToHost, s_out));
            }
        }
        // the count is complete once the kernels of the last chunk have run (stream order on s_k)
        if (update) RBG_CUDA(h, cudaMemcpyAsync(&neg_count, h->scratch_flag, sizeof(int), cudaMemcpyDeviceToHost, s_k));
        return RBG_OK;
    };
    const int rc = pipeline();
    const cudaError_t d_out = cudaStreamSynchronize(s_out), d_k = cudaStreamSynchronize(s_k), d_in = cudaStreamSynchronize(s_in);
    if (rc != RBG_OK) return rc;                       // the pipeline's own message stands
    RBG_CUDA(h, d_out); RBG_CUDA(h, d_k); RBG_CUDA(h, d_in);
    if (update) *neg_count_host = neg_count;
    return RBG_OK;
}

int rbg_collision_host(rbg_handle* h, const double* f_host, double* C_host, int n_samples, uint64_t seed) {
    return host_sweep(h, f_host, C_host, false, 0.0, nullptr, n_samples, seed);
}

int rbg_collision_update_host(rbg_handle* h, const double* f_host, double* f_out_host, double dt, int* neg_count_host,
                              int n_samples, uint64_t seed) {
    return host_sweep(h, f_host, f_out_host, true, dt, neg_count_host, n_samples, seed);
}

size_t rbg_f_elems(const rbg_handle* h) { return h ? h->f_elems : 0; }
int rbg_n_roles(const rbg_handle* h) { return h ? (int)h->roles.size() : 0; }
int rbg_role_info(const rbg_handle* h, int r, int species[4], double* sym, double* cl, double* cg, int* process) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (r < 0 || r >= (int)h->roles.size()) { h->err = "rbg_role_info: role index out of range"; return RBG_E_INVALID_ARG; }
    const Role& R = h->roles[r];
    if (species) for (int i = 0; i < 4; ++i) species[i] = R.s[i];
    if (sym) *sym = R.sym;
    if (cl) *cl = R.cl;
    if (cg) *cg = R.cg;
    if (process) *process = R.process;
    return RBG_OK;
}
uint64_t rbg_sample_evals(const rbg_handle* h, int n_samples) {
    if (!h) return 0;
    uint64_t t = 0;
    for (const Role& r : h->roles) t += (uint64_t)h->nx * h->np[r.s[0]] * (uint64_t)n_samples;
    return t;
}
int rbg_last_launch_count(const rbg_handle* h) { return h ? h->last_launches : 0; }

int rbg_set_option(rbg_handle* h, const char* key, int value) {
    if (!h || !key) return fail(h, RBG_E_INVALID_ARG, "null argument");
    const std::string k(key);
    if (k == "warps_per_cta") { if (value < 0 || value > 32) return fail(h, RBG_E_INVALID_ARG, "warps_per_cta must be 0 (auto) or 1..32"); h->opt_warps = value; }
    else if (k == "samples_per_lane") { if (value < 0 || value > 2) return fail(h, RBG_E_INVALID_ARG, "samples_per_lane must be 0 (auto), 1 or 2"); h->opt_spl = value; }
    else if (k == "p1_per_cta") { if (value < 0) return fail(h, RBG_E_INVALID_ARG, "p1_per_cta must be >= 0 (0 = auto)"); h->opt_p1_per_cta = value; }
#ifdef RBG_CHECKED
    else if (k == "selfcheck_probe") {             // checked build only: `value` threads fail one check of every class
        if (value < 0 || value > 1024) return fail(h, RBG_E_INVALID_ARG, "selfcheck_probe must be 0..1024");
        DeviceGuard guard(h->device);
        rbg::selfcheck_probe_kernel<<<1, 1024>>>(value);
        RBG_CUDA(h, cudaDeviceSynchronize());
    }
#endif
    else if (k == "sym_tables") { if (value < 0 || value > 1) return fail(h, RBG_E_INVALID_ARG, "sym_tables must be 0 (global atomics) or 1 (shared-memory accumulator tables)"); h->opt_sym_tables = value; }
    else if (k == "vlasov_path") { if (value < 0 || value > 1) return fail(h, RBG_E_INVALID_ARG, "vlasov_path must be 0 (auto) or 1 (general staged kernel)"); h->opt_vlasov_path = value; }
    else if (k == "moments_path") { if (value < 0 || value > 1) return fail(h, RBG_E_INVALID_ARG, "moments_path must be 0 (auto) or 1 (general staged kernel)"); h->opt_moments_path = value; }
    else if (k == "gather") { if (value < 0 || value > 2) return fail(h, RBG_E_INVALID_ARG, "gather must be 0, 1 or 2"); h->opt_gather = value; }
    else return fail(h, RBG_E_INVALID_ARG, "unknown option " + k);
    return RBG_OK;
}

const char* rbg_last_error(const rbg_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

void rbg_destroy(rbg_handle* h) {
    if (!h) return;
    DeviceGuard guard(h->device);
    cudaFree(h->scratch_f); cudaFree(h->scratch_c); cudaFree(h->scratch_flag);
    for (cudaStream_t st : h->host_streams) if (st) cudaStreamDestroy(st);
    for (cudaEvent_t ev : h->host_events) if (ev) cudaEventDestroy(ev);
    for (double* p : h->tab_iE) cudaFree(p);
    for (double* p : h->tab_v) cudaFree(p);
    cudaFree(h->charges_dev);
    cudaFree(h->dir_tab);
    delete h;
}

// ---- NEXT-4: the steps either side of the collision term -------------------------------------------------------
namespace {
rbg::SpeciesTables species_tables(const rbg_handle* h, int s) {
    rbg::SpeciesTables t;
    t.iE = h->tab_iE[s]; t.v = h->tab_v[s];
    for (int d = 0; d < 3; ++d) {
        t.pmin[d] = h->grids[s].pmin[d];
        t.delta[d] = (h->grids[s].pmax[d] - h->grids[s].pmin[d]) / (double)h->grids[s].n[d];
        t.n[d] = h->grids[s].n[d];
    }
    t.np = (int)h->np[s];
    t.mass = h->species[s].mass; t.charge = h->species[s].charge;
    return t;
}
}  // namespace

namespace {
// Geometry of the persistent staged kernels (moments, Vlasov): shared memory is [head][1/E table][ring of stages].  A
// stage is `group` consecutive spatial cells: at least one per team, an even number when np is odd (so that its byte
// count is a multiple of 16), and 32 KB or more per copy where the domain allows it.
struct StagedGeometry { int team, group, n_stages, lead, ctas; size_t smem; bool ok; };
StagedGeometry staged_geometry(const rbg_handle* h, int s, const double* fs, size_t head, bool table_in_smem) {
    StagedGeometry g{};
    const size_t np = h->np[s];
    const int nyz = h->grids[s].n[1] * h->grids[s].n[2];
    const size_t tab_bytes = table_in_smem ? (np * 8 + 127) & ~(size_t)127 : 0;
    const size_t avail = (size_t)h->max_smem_optin > head + tab_bytes ? (size_t)h->max_smem_optin - head - tab_bytes : 0;
    g.team = 32;
    while (g.team < rbg::MOM_THREADS && g.team < nyz) g.team *= 2;
    g.group = rbg::MOM_THREADS / g.team;
    if ((np % 2) && (g.group % 2)) g.group *= 2;
    while ((size_t)g.group * np * 8 < 32768 && (size_t)(2 * g.group) * np * 8 * 3 <= avail) g.group *= 2;
    while (g.group > 1 && (size_t)g.group * np * 8 * 2 > avail) g.group /= 2;
    if (g.group < rbg::MOM_THREADS / g.team) g.team = rbg::MOM_THREADS / g.group;          // fewer, larger teams
    const size_t stage_bytes = ((size_t)g.group * np * 8 + 127) & ~(size_t)127;
    g.n_stages = (int)std::min<size_t>(rbg::MOM_MAX_STAGES, avail / stage_bytes);
    g.ok = g.n_stages >= 2;
    // an odd leading cell puts the groups on 16-byte boundaries when the species block starts 8 bytes off one
    g.lead = (reinterpret_cast<uintptr_t>(fs) % 16 != 0 && (np % 2)) ? 1 : 0;
    g.smem = head + tab_bytes + (size_t)g.n_stages * stage_bytes;
    const int n_units = (g.lead ? 1 : 0) + (h->nx - g.lead + g.group - 1) / g.group;
    g.ctas = std::max(1, std::min(h->sm_count, n_units));
    return g;
}
}  // namespace

int rbg_moments(rbg_handle* h, const double* f_dev, double* M_dev, double* total_dev, double* em_dev, void* cuda_stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f_dev || !M_dev) return fail(h, RBG_E_INVALID_ARG, "null buffer");
    {
        const size_t fb = h->f_elems * sizeof(double), cellb = (size_t)h->nx * rbg::N_MOMENTS * sizeof(double);
        if (ranges_overlap(f_dev, fb, M_dev, (size_t)h->n_species * cellb) || (total_dev && ranges_overlap(f_dev, fb, total_dev, cellb)) ||
            (em_dev && ranges_overlap(f_dev, fb, em_dev, (size_t)h->nx * 4 * sizeof(double))))
            return fail(h, RBG_E_INVALID_ARG, "an output buffer of rbg_moments overlaps f_dev");
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(h->device);
    h->last_launches = 0;
    for (int s = 0; s < h->n_species; ++s) {
        const rbg::SpeciesTables tb = species_tables(h, s);
        const double* fs = f_dev + h->sp_off[s];
        double* Ms = M_dev + (size_t)s * h->nx * rbg::N_MOMENTS;
        const int nyz = tb.n[1] * tb.n[2];
        // head: mbarriers, counters, MOM_RED reduction buffers, p_x table
        const size_t head = (128 + ((size_t)rbg::MOM_RED * (rbg::MOM_THREADS / 32) * 16 + (size_t)tb.n[0]) * 8 + 127) & ~(size_t)127;
        // Momentum grid symmetric about 0 in every direction, at most 512 (p_y, p_z) columns, a cell of whole 16-byte units
        // that fits three times next to the octant table: moments_sym_kernel (rbg_be_kernels.cuh)
        {
            bool sym = h->opt_moments_path != 1 && nyz <= rbg::MS_TEAM * rbg::MS_MAXC && (tb.np * 8) % 16 == 0 &&
                       reinterpret_cast<uintptr_t>(fs) % 16 == 0;
            for (int d = 0; d < 3; ++d) {
                const rbg_momentum_grid& G = h->grids[s];
                sym = sym && std::fabs(G.pmin[d] + G.pmax[d]) <= 1e-12 * (G.pmax[d] - G.pmin[d]);
            }
            const int c0 = tb.n[0] / 2, n0h = (tb.n[0] + 1) / 2, n1h = (tb.n[1] + 1) / 2, n2h = (tb.n[2] + 1) / 2;
            const size_t head_sym = (128 + ((size_t)rbg::MS_STAGES * (rbg::MS_TEAM / 32) * 16 + 2 * (size_t)c0 + (size_t)n0h * n1h * n2h) * 8 + 127) & ~(size_t)127;
            const size_t smem_sym = head_sym + (size_t)rbg::MS_STAGES * (((size_t)tb.np * 8 + 127) & ~(size_t)127);
            if (sym && smem_sym <= (size_t)h->max_smem_optin) {
                RBG_CUDA(h, ensure_max_smem(rbg::moments_sym_kernel, h->device, h->max_smem_optin));
                rbg::moments_sym_kernel<<<std::max(1, std::min(h->sm_count, h->nx)), rbg::MS_THREADS, smem_sym, st>>>(fs, tb, h->nx, Ms);
                RBG_CUDA(h, cudaGetLastError());
                ++h->last_launches;
                continue;
            }
        }
        // the 1/E table lives in shared memory when it fits next to two stages (measured: reading it through L1 and
        // spending its shared memory on a third stage is slower, 0.73 vs 0.58 ms on config 4: the kernel is bound by the
        // CTA's own instruction latency, the two-stage ring alone streams at 6.2 TB/s); otherwise it is read through L1
        bool ie_smem = true;
        StagedGeometry g = staged_geometry(h, s, fs, head, true);
        if (!g.ok) { ie_smem = false; g = staged_geometry(h, s, fs, head, false); }
        if (!g.ok) {                                   // the block does not fit twice: read f straight from global memory
            rbg::moments_direct_kernel<<<h->nx, 128, 0, st>>>(fs, tb, h->nx, Ms);
            RBG_CUDA(h, cudaGetLastError());
            ++h->last_launches;
            continue;
        }
        const bool one_team = g.team == rbg::MOM_THREADS && g.n_stages * g.group <= rbg::MOM_RED;
        auto launch = [&](auto kern) -> cudaError_t {
            const cudaError_t e = ensure_max_smem(kern, h->device, h->max_smem_optin);
            if (e != cudaSuccess) return e;
            kern<<<g.ctas, rbg::MOM_THREADS, g.smem, st>>>(fs, tb, h->nx, Ms, g.group, g.n_stages, g.team, g.lead);
            return cudaSuccess;
        };
        if (one_team) {
            if (g.team >= nyz) RBG_CUDA(h, ie_smem ? launch(rbg::moments_kernel<1, true, true>) : launch(rbg::moments_kernel<1, false, true>));
            else               RBG_CUDA(h, ie_smem ? launch(rbg::moments_kernel<4, true, true>) : launch(rbg::moments_kernel<4, false, true>));
        } else {
            if (g.team >= nyz) RBG_CUDA(h, ie_smem ? launch(rbg::moments_kernel<1, true, false>) : launch(rbg::moments_kernel<1, false, false>));
            else               RBG_CUDA(h, ie_smem ? launch(rbg::moments_kernel<4, true, false>) : launch(rbg::moments_kernel<4, false, false>));
        }
        RBG_CUDA(h, cudaGetLastError());
        ++h->last_launches;
    }
    if (total_dev || em_dev) {
        const size_t n = (size_t)h->nx * rbg::N_MOMENTS;
        rbg::totals_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(M_dev, h->charges_dev, h->n_species, h->nx, total_dev, em_dev);
        RBG_CUDA(h, cudaGetLastError());
        ++h->last_launches;
    }
    return RBG_OK;
}

}  // extern "C" (re-opened below)

// ---- rbg_moments_static: the moments of one species for callers that must not allocate device memory -----------------
// Everything this entry point needs besides the caller's f and M is the species' 1/E_p table, and that lives here, in the
// library image, instead of in a cudaMalloc'ed buffer.  Every GPU that loads the library carries these 512 KB until the
// process exits; every call shares them.
//
// In host code `g_static_inv_energy` is NOT a device address: it names a host-side shadow the runtime uses as a lookup
// key.  Handing it to a kernel would make the kernel read and write wherever that host address happens to point.  The
// address a kernel may use is per device and comes from cudaGetSymbolAddress, asked for once per device with that device
// current (static_table_for_current_device below).
static __device__ __align__(256) double g_static_inv_energy[RBG_MOMENTS_STATIC_MAX_CELLS];

namespace {

// 1/E_p of every momentum-cell centre, the same roundings in the same order as the host loop of rbg_create (this file is
// compiled with -fmad=false, and the double-precision sqrt and divide of the device are correctly rounded), so the table
// holds the bits rbg_create would have uploaded.  Every entry in [0, n0 n1 n2) is overwritten: nothing is assumed about
// what the previous call left in the array.
__global__ void __launch_bounds__(256)
inv_energy_fill_kernel(double* __restrict__ table, int n0, int n1, int n2, double pmin0, double pmin1, double pmin2,
                       double delta0, double delta1, double delta2, double msq) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int nyz = n1 * n2;
    if (j >= n0 * nyz) return;
    const int i0 = j / nyz, r = j - i0 * nyz, i1 = r / n2, i2 = r - i1 * n2;
    const double px = rbg::cell_centre(i0, delta0, pmin0);
    const double py = rbg::cell_centre(i1, delta1, pmin1);
    const double pz = rbg::cell_centre(i2, delta2, pmin2);
    const double E = sqrt(((px * px + py * py) + pz * pz) + msq);
    table[j] = E > 0.0 ? 1.0 / E : 0.0;
}

// Device address of g_static_inv_energy on the CURRENT device, looked up on the first call made with that device current
// and remembered.  cudaGetSymbolAddress initialises the context / loads this module on the device if that has not happened
// yet, which is why the first call belongs in the caller's set-up phase and outside any stream capture.
enum { STATIC_MAX_DEVICES = 64 };
std::mutex g_static_mu;
double* g_static_table[STATIC_MAX_DEVICES] = {};

int static_table_for_current_device(double** table) {
    int dev = -1;
    RBG_CUDA(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES)
        return fail(nullptr, RBG_E_UNSUPPORTED, "rbg_moments_static: device ordinal " + std::to_string(dev) + " is beyond the " +
                                                std::to_string((int)STATIC_MAX_DEVICES) + " this entry point keeps an address for");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_table[dev]) {
        void* p = nullptr;
        RBG_CUDA(nullptr, cudaGetSymbolAddress(&p, g_static_inv_energy));
        if (!p) return fail(nullptr, RBG_E_CUDA, "rbg_moments_static: cudaGetSymbolAddress returned a null address");
        g_static_table[dev] = static_cast<double*>(p);
    }
    *table = g_static_table[dev];
    return RBG_OK;
}

}  // namespace

extern "C" {

int rbg_moments_static(const rbg_momentum_grid* grid, double mass, int n_cells, const double* f_dev, double* M_dev,
                       void* cuda_stream) {
    if (!grid || !f_dev || !M_dev) return fail(nullptr, RBG_E_INVALID_ARG, "rbg_moments_static: null argument");
    if (!(mass >= 0.0)) return fail(nullptr, RBG_E_INVALID_ARG, "rbg_moments_static: negative mass");
    if (n_cells < 0) return fail(nullptr, RBG_E_INVALID_ARG, "rbg_moments_static: n_cells must be >= 0");
    double cells = 1.0;
    for (int d = 0; d < 3; ++d) {
        if (grid->n[d] <= 0) return fail(nullptr, RBG_E_INVALID_ARG, "rbg_moments_static: momentum grid counts must be positive");
        if (!(grid->pmax[d] > grid->pmin[d])) return fail(nullptr, RBG_E_INVALID_ARG, "rbg_moments_static: pmax must exceed pmin");
        cells *= (double)grid->n[d];
    }
    if (cells > (double)RBG_MOMENTS_STATIC_MAX_CELLS)
        return fail(nullptr, RBG_E_UNSUPPORTED,
                    "rbg_moments_static: the momentum grid has " + std::to_string((long long)cells) + " cells, the built-in table holds " +
                    std::to_string((int)RBG_MOMENTS_STATIC_MAX_CELLS) +
                    " (RBG_MOMENTS_STATIC_MAX_CELLS); larger grids need rbg_create + rbg_moments, which allocate");
    if (n_cells == 0) return RBG_OK;
    if (ranges_overlap(f_dev, (size_t)n_cells * (size_t)cells * sizeof(double), M_dev, (size_t)n_cells * rbg::N_MOMENTS * sizeof(double)))
        return fail(nullptr, RBG_E_INVALID_ARG, "rbg_moments_static: M_dev overlaps f_dev");
    double* table = nullptr;
    const int rc = static_table_for_current_device(&table);
    if (rc != RBG_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    rbg::SpeciesTables tb;
    std::memset(&tb, 0, sizeof tb);
    for (int d = 0; d < 3; ++d) {
        tb.pmin[d] = grid->pmin[d];
        tb.delta[d] = (grid->pmax[d] - grid->pmin[d]) / (double)grid->n[d];
        tb.n[d] = grid->n[d];
    }
    tb.np = (int)cells;
    tb.mass = mass;
    tb.iE = table;                 // the device address, never the symbol
    tb.v = nullptr;                // the moment sums do not read the velocity table
    inv_energy_fill_kernel<<<(tb.np + 255) / 256, 256, 0, st>>>(table, tb.n[0], tb.n[1], tb.n[2], tb.pmin[0], tb.pmin[1], tb.pmin[2],
                                                                tb.delta[0], tb.delta[1], tb.delta[2], mass * mass);
    RBG_CUDA(nullptr, cudaGetLastError());
    rbg::moments_direct_kernel<<<n_cells, 128, 0, st>>>(f_dev, tb, n_cells, M_dev);
    RBG_CUDA(nullptr, cudaGetLastError());
    return RBG_OK;
}

int rbg_drift_step(rbg_handle* h, const double* f_dev, double* f_out_dev, const rbg_drift_params* p, void* cuda_stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f_dev || !f_out_dev || !p) return fail(h, RBG_E_INVALID_ARG, "null argument");
    if (ranges_overlap(f_dev, h->f_elems * sizeof(double), f_out_dev, h->f_elems * sizeof(double)))
        return fail(h, RBG_E_INVALID_ARG, "f_out_dev overlaps f_dev (the stencil reads neighbours)");
    if (!(p->dt >= 0.0)) return fail(h, RBG_E_INVALID_ARG, "dt must be >= 0");
    if (h->ix_offset != 0) return fail(h, RBG_E_UNSUPPORTED, "the drift stencil needs the whole spatial domain on one GPU (no ghost-layer exchange)");
    rbg::DriftParams dp;
    dp.dt = p->dt; dp.zeta = p->zeta;
    for (int d = 0; d < 3; ++d) {
        if (!(p->dx[d] > 0.0)) return fail(h, RBG_E_INVALID_ARG, "dx must be positive");
        if (p->bc[d] != 0 && p->bc[d] != 1) return fail(h, RBG_E_INVALID_ARG, "bc must be 0 (wall) or 1 (periodic)");
        dp.inv_dx[d] = 1.0 / p->dx[d]; dp.nxyz[d] = h->nxyz[d]; dp.bc[d] = p->bc[d];
    }
    if (!(p->zeta >= 0.0 && p->zeta <= 1.0)) return fail(h, RBG_E_INVALID_ARG, "zeta must be in [0, 1]");
    if (p->zeta != 0.0)
        for (int s = 0; s < h->n_species; ++s)
            for (int d = 0; d < 3; ++d)
                if (p->bc[d] == 0 && std::fabs(h->grids[s].pmin[d] + h->grids[s].pmax[d]) > 1e-12 * (h->grids[s].pmax[d] - h->grids[s].pmin[d]))
                    return fail(h, RBG_E_UNSUPPORTED, "reflecting walls need momentum grids symmetric about 0 (the mirrored momentum must be a grid cell)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(h->device);
    h->last_launches = 0;
    dp.zseg = std::min(16, h->nxyz[2]);                 // measured on config 4: segments of 8 or 32 cells are slower
    dp.tile_y = std::min(8, h->nxyz[1]);                // measured on config 4: tiles of 2, 4 or 16 rows are slower
    const long nzseg = (h->nxyz[2] + dp.zseg - 1) / dp.zseg, nyt = (h->nxyz[1] + dp.tile_y - 1) / dp.tile_y;
    for (int s = 0; s < h->n_species; ++s) {
        const long nchunks = ((long)h->np[s] + 255) / 256;
        const long grid = nchunks * nzseg * dp.tile_y * h->nxyz[0] * nyt;
        if (grid > 0x7fffffffL) return fail(h, RBG_E_UNSUPPORTED, "rbg_drift_step: grid too large");
        rbg::drift_upfd_kernel<<<(unsigned)grid, 256, 0, st>>>(f_dev + h->sp_off[s], f_out_dev + h->sp_off[s], species_tables(h, s), dp);
        RBG_CUDA(h, cudaGetLastError());
        ++h->last_launches;
    }
    return RBG_OK;
}

int rbg_drift_step_pfl(rbg_handle* h, const double* f_dev, double* f_out_dev, double dt, const double* dx, void* cuda_stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f_dev || !f_out_dev || !dx) return fail(h, RBG_E_INVALID_ARG, "null argument");
    if (ranges_overlap(f_dev, h->f_elems * sizeof(double), f_out_dev, h->f_elems * sizeof(double)))
        return fail(h, RBG_E_INVALID_ARG, "f_out_dev overlaps f_dev (the stencil reads neighbours)");
    if (!(dt >= 0.0)) return fail(h, RBG_E_INVALID_ARG, "dt must be >= 0");
    if (h->ix_offset != 0) return fail(h, RBG_E_UNSUPPORTED, "the drift stencil needs the whole spatial domain on one GPU (no ghost-layer exchange)");
    rbg::DriftParams dp;
    dp.dt = dt; dp.zeta = 0.0;
    for (int d = 0; d < 3; ++d) {
        if (!(dx[d] > 0.0)) return fail(h, RBG_E_INVALID_ARG, "dx must be positive");
        dp.inv_dx[d] = 1.0 / dx[d]; dp.nxyz[d] = h->nxyz[d]; dp.bc[d] = 1;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(h->device);
    h->last_launches = 0;
    dp.zseg = std::min(16, h->nxyz[2]);
    dp.tile_y = std::min(8, h->nxyz[1]);
    const long nzseg = (h->nxyz[2] + dp.zseg - 1) / dp.zseg, nyt = (h->nxyz[1] + dp.tile_y - 1) / dp.tile_y;
    for (int s = 0; s < h->n_species; ++s) {
        const long nchunks = ((long)h->np[s] + 255) / 256;
        const long grid = nchunks * nzseg * dp.tile_y * h->nxyz[0] * nyt;
        if (grid > 0x7fffffffL) return fail(h, RBG_E_UNSUPPORTED, "rbg_drift_step_pfl: grid too large");
        rbg::drift_pfl_kernel<<<(unsigned)grid, 256, 0, st>>>(f_dev + h->sp_off[s], f_out_dev + h->sp_off[s], species_tables(h, s), dp);
        RBG_CUDA(h, cudaGetLastError());
        ++h->last_launches;
    }
    return RBG_OK;
}

int rbg_vlasov_step(rbg_handle* h, const double* f_dev, double* f_out_dev, double dt, const double* E_dev, const double* B_dev,
                    void* cuda_stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f_dev || !f_out_dev || !E_dev || !B_dev) return fail(h, RBG_E_INVALID_ARG, "null buffer");
    if (ranges_overlap(f_dev, h->f_elems * sizeof(double), f_out_dev, h->f_elems * sizeof(double)))
        return fail(h, RBG_E_INVALID_ARG, "f_out_dev overlaps f_dev (the stencil reads neighbours)");
    if (!(dt >= 0.0)) return fail(h, RBG_E_INVALID_ARG, "dt must be >= 0");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DeviceGuard guard(h->device);
    h->last_launches = 0;
    rbg::VlasovParams vp;
    vp.dt = dt; vp.nx_cells = h->nx; vp.E = E_dev; vp.B = B_dev;
    for (int s = 0; s < h->n_species; ++s) {
        const rbg::SpeciesTables tb = species_tables(h, s);
        const double* fs = f_dev + h->sp_off[s];
        double* os = f_out_dev + h->sp_off[s];
        const int nyz = tb.n[1] * tb.n[2];
        // Momentum grid symmetric about 0 in every direction, at most 800 (p_y, p_z) columns, a cell of whole 16-byte units
        // that fits three times next to the octant table: vlasov_sym_kernel (rbg_be_kernels.cuh)
        {
            bool sym = h->opt_vlasov_path != 1 && nyz <= rbg::VS_MAX_THREADS && nyz % 2 == 0 &&          // planes of whole 16-byte units
                       reinterpret_cast<uintptr_t>(fs) % 16 == 0;
            for (int d = 0; d < 3; ++d) {
                const rbg_momentum_grid& G = h->grids[s];
                sym = sym && std::fabs(G.pmin[d] + G.pmax[d]) <= 1e-12 * (G.pmax[d] - G.pmin[d]);
            }
            const int n0h = (tb.n[0] + 1) / 2, n1h = (tb.n[1] + 1) / 2, n2h = (tb.n[2] + 1) / 2;
            const size_t head_sym = (128 + (size_t)tb.n[0] * 16 + (size_t)n0h * n1h * n2h * 8 + 127) & ~(size_t)127;
            // a stage holds the cell plus one halo plane on either side (the periodic p_x neighbours)
            const size_t smem_sym = head_sym + (size_t)rbg::VS_STAGES * (((size_t)tb.np * 8 + 2 * (size_t)nyz * 8 + 127) & ~(size_t)127);
            if (sym && smem_sym <= (size_t)h->max_smem_optin) {
                // segments per column: as many as fit in 800 threads, each of ceil(n0 / segs) planes
                int segs = std::max(1, std::min(tb.n[0], rbg::VS_MAX_THREADS / nyz));
                const int seg_len = (tb.n[0] + segs - 1) / segs;
                segs = (tb.n[0] + seg_len - 1) / seg_len;
                const int threads = ((segs * nyz + 31) / 32) * 32;
                RBG_CUDA(h, ensure_max_smem(rbg::vlasov_sym_kernel, h->device, h->max_smem_optin));
                rbg::vlasov_sym_kernel<<<std::max(1, std::min(h->sm_count, h->nx)), threads, smem_sym, st>>>(fs, os, tb, vp, segs, seg_len);
                RBG_CUDA(h, cudaGetLastError());
                ++h->last_launches;
                continue;
            }
        }
        const size_t head = (128 + (size_t)tb.n[0] * 8 + 127) & ~(size_t)127;
        const StagedGeometry g = staged_geometry(h, s, fs, head, true);
        if (!g.ok) {                                   // the block does not fit twice next to the table: direct kernel
            const int slab = 16, nchunks = (tb.np + 255) / 256;
            const long grid = (long)nchunks * ((h->nx + slab - 1) / slab);
            rbg::vlasov_direct_kernel<<<(unsigned)grid, 256, 0, st>>>(fs, os, tb, vp, slab);
            RBG_CUDA(h, cudaGetLastError());
            ++h->last_launches;
            continue;
        }
        if (g.team >= nyz) {
            RBG_CUDA(h, ensure_max_smem(rbg::vlasov_upfd_kernel<1>, h->device, h->max_smem_optin));
            rbg::vlasov_upfd_kernel<1><<<g.ctas, rbg::MOM_THREADS, g.smem, st>>>(fs, os, tb, vp, g.group, g.n_stages, g.team, g.lead);
        } else {
            RBG_CUDA(h, ensure_max_smem(rbg::vlasov_upfd_kernel<4>, h->device, h->max_smem_optin));
            rbg::vlasov_upfd_kernel<4><<<g.ctas, rbg::MOM_THREADS, g.smem, st>>>(fs, os, tb, vp, g.group, g.n_stages, g.team, g.lead);
        }
        RBG_CUDA(h, cudaGetLastError());
        ++h->last_launches;
    }
    return RBG_OK;
}

int rbg_be_step(rbg_handle* h, double* f_dev, double* scratch_dev, const rbg_be_step_params* p, const double* E_dev,
                const double* B_dev, int* neg_flag_dev, void* cuda_stream) {
    if (!h) return fail(nullptr, RBG_E_INVALID_ARG, "null handle");
    if (!f_dev || !scratch_dev || !p) return fail(h, RBG_E_INVALID_ARG, "null argument");
    const size_t bytes = h->f_elems * sizeof(double);
    if (ranges_overlap(f_dev, bytes, scratch_dev, bytes)) return fail(h, RBG_E_INVALID_ARG, "scratch_dev overlaps f_dev");
    if (p->do_vlasov && (!E_dev || !B_dev)) return fail(h, RBG_E_INVALID_ARG, "do_vlasov needs E_dev and B_dev");
    if (p->do_collision && !neg_flag_dev) return fail(h, RBG_E_INVALID_ARG, "do_collision needs neg_flag_dev");
    // everything the sub-steps would refuse is refused here, before the first launch touches f_dev
    if (p->do_collision != 0 && p->do_collision != 1 && p->do_collision != 2) return fail(h, RBG_E_INVALID_ARG, "do_collision must be 0, 1 or 2");
    if (p->do_collision && p->n_samples <= 0) return fail(h, RBG_E_INVALID_ARG, "n_samples must be positive");
    if (p->do_collision == 2) {
        if (h->flags & RBG_FP32_KINEMATICS) return fail(h, RBG_E_UNSUPPORTED, "rbg_collision_symmetric is fp64 only");
        for (const Role& r : h->roles)
            if (r.sampler != RBG_SAMPLER_UNIFORM) return fail(h, RBG_E_UNSUPPORTED, "rbg_collision_symmetric supports the uniform sampler only");
    }
    if ((p->do_drift || p->do_vlasov) && !(p->dt >= 0.0)) return fail(h, RBG_E_INVALID_ARG, "dt must be >= 0");
    if (p->do_drift) {
        if (h->ix_offset != 0) return fail(h, RBG_E_UNSUPPORTED, "the drift stencil needs the whole spatial domain on one GPU (no ghost-layer exchange)");
        if (!(p->zeta >= 0.0 && p->zeta <= 1.0)) return fail(h, RBG_E_INVALID_ARG, "zeta must be in [0, 1]");
        for (int d = 0; d < 3; ++d) {
            if (!(p->dx[d] > 0.0)) return fail(h, RBG_E_INVALID_ARG, "dx must be positive");
            if (p->bc[d] != 0 && p->bc[d] != 1) return fail(h, RBG_E_INVALID_ARG, "bc must be 0 (wall) or 1 (periodic)");
        }
        if (p->zeta != 0.0)
            for (int s = 0; s < h->n_species; ++s)
                for (int d = 0; d < 3; ++d)
                    if (p->bc[d] == 0 && std::fabs(h->grids[s].pmin[d] + h->grids[s].pmax[d]) > 1e-12 * (h->grids[s].pmax[d] - h->grids[s].pmin[d]))
                        return fail(h, RBG_E_UNSUPPORTED, "reflecting walls need momentum grids symmetric about 0 (the mirrored momentum must be a grid cell)");
    }
    DeviceGuard guard(h->device);
    double *cur = f_dev, *nxt = scratch_dev;
    int launches = 0, rc;
    if (p->do_drift) {
        rbg_drift_params dp;
        dp.dt = p->dt; dp.zeta = p->zeta;
        for (int d = 0; d < 3; ++d) { dp.dx[d] = p->dx[d]; dp.bc[d] = p->bc[d]; }
        if ((rc = rbg_drift_step(h, cur, nxt, &dp, cuda_stream)) != RBG_OK) return rc;
        launches += h->last_launches; std::swap(cur, nxt);
    }
    if (p->do_vlasov) {
        if ((rc = rbg_vlasov_step(h, cur, nxt, p->dt, E_dev, B_dev, cuda_stream)) != RBG_OK) return rc;
        launches += h->last_launches; std::swap(cur, nxt);
    }
    if (p->do_collision == 2) {
        // conservative estimator: C into the free buffer, then cur += 3 dt C in place
        if ((rc = rbg_collision_symmetric(h, cur, nxt, p->n_samples, p->seed, cuda_stream)) != RBG_OK) return rc;
        launches += h->last_launches;
        rbg::axpy_count_kernel<<<h->sm_count * 8, 256, 0, (cudaStream_t)cuda_stream>>>(cur, nxt, 3.0 * p->dt, h->f_elems, neg_flag_dev);
        RBG_CUDA(h, cudaGetLastError());
        ++launches;
    } else if (p->do_collision) {
        if ((rc = run(h, cur, nxt, true, 3.0 * p->dt, neg_flag_dev, p->n_samples, p->seed, cuda_stream)) != RBG_OK) return rc;
        launches += h->last_launches; std::swap(cur, nxt);
    }
    if (cur != f_dev) RBG_CUDA(h, cudaMemcpyAsync(f_dev, cur, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    h->last_launches = launches;
    return RBG_OK;
}

int rbg_selfcheck_failures(uint64_t* counts) {
    if (!counts) return fail(nullptr, RBG_E_INVALID_ARG, "null argument");
#ifdef RBG_CHECKED
    unsigned long long h[rbg::CHK_CLASSES];
    RBG_CUDA(nullptr, cudaDeviceSynchronize());
    RBG_CUDA(nullptr, cudaMemcpyFromSymbol(h, rbg::g_check_failures, sizeof h));
    for (int i = 0; i < rbg::CHK_CLASSES; ++i) counts[i] = h[i];
    return RBG_OK;
#else
    for (int i = 0; i < rbg::CHK_CLASSES; ++i) counts[i] = 0;
    return fail(nullptr, RBG_E_UNSUPPORTED, "not a checked build (python -m paper_2308_04869_b200.build --checked)");
#endif
}

int rbg_selftest_math(uint64_t n_operands, uint32_t seed, uint64_t* mismatches) {
    if (!mismatches) return fail(nullptr, RBG_E_INVALID_ARG, "null argument");
    unsigned long long* d = nullptr;
    RBG_CUDA(nullptr, cudaMalloc(&d, 8));
    RBG_CUDA(nullptr, cudaMemset(d, 0, 8));
    const int ctas = 592, threads = 256;
    const unsigned long long per = (n_operands + (uint64_t)ctas * threads - 1) / ((uint64_t)ctas * threads);
    rbg::math_selftest_kernel<<<ctas, threads>>>(per, seed, d);
    cudaError_t e = cudaDeviceSynchronize();
    unsigned long long hbad = 0;
    if (e == cudaSuccess) e = cudaMemcpy(&hbad, d, 8, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return fail(nullptr, RBG_E_CUDA, cudaGetErrorString(e));
    *mismatches = hbad;
    return RBG_OK;
}

int rbg_probe_alu_peak(int what, int iters, double* ops_per_s, void* cuda_stream) {
    if (!ops_per_s || iters <= 0 || what < 0 || what > 4) return fail(nullptr, RBG_E_INVALID_ARG, "bad probe arguments");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    RBG_CUDA(nullptr, cudaGetDevice(&dev));
    RBG_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int ctas = sms * 8, threads = 256;
    void* buf = nullptr;
    RBG_CUDA(nullptr, cudaMalloc(&buf, (size_t)ctas * threads * 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {            // rep 0 warms clocks and instruction cache
        cudaEventRecord(e0, st);
        if (what == 0) rbg::alu_probe_kernel<double><<<ctas, threads, 0, st>>>((double*)buf, 1.0000001, 1e-9, iters);
        else if (what == 1) rbg::alu_probe_kernel<float><<<ctas, threads, 0, st>>>((float*)buf, 1.0000001f, 1e-9f, iters);
        else if (what == 2) rbg::alu_probe_kernel<unsigned><<<ctas, threads, 0, st>>>((unsigned*)buf, 2654435761u, 12345u, iters);
        else if (what == 3) rbg::dfma3_probe_kernel<<<ctas, threads, 0, st>>>((double*)buf, iters);
        else rbg::widemul_probe_kernel<<<ctas, threads, 0, st>>>((unsigned*)buf, iters);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(buf); return fail(nullptr, RBG_E_CUDA, cudaGetErrorString(e)); }
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf);
    *ops_per_s = (double)ctas * threads * 8.0 * (double)iters / (best * 1e-3);
    return RBG_OK;
}

}  // extern "C"
