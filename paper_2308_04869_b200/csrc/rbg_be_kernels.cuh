// rbg_be_kernels.cuh -- sm_100a device code for the steps either side of the collision term:
//   moments_kernel      n_a, j_a (Eq. 5-6), T^{mu nu}_a (Eq. 9)
//   totals_kernel       sums over species (Eq. 7, 9) and rho, J (Eq. 15)
//   drift_upfd_kernel   first-order UPFD step of the drift term (Eq. 25, 28-30)
//   vlasov_upfd_kernel  first-order UPFD step of the Vlasov term (Eq. 26, 34)
// All three are HBM-bound streaming kernels (8 B read per phase-space cell for the moments, 8 B read + 8 B written for
// the two stencils); their arithmetic is kept below the memory time by hoisting everything that depends only on the
// momentum cell out of the loop over spatial cells (stencils) or out of the loop over p_x (moments).
// hbar = c = 1.  Layout of f: [species][ix][ipx][ipy][ipz], ix = (i_x ny + i_y) nz + i_z.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rbg {

// Checked build: a warp that consumes a ring slot verifies, before its first and after its last read, that the slot still
// holds the unit it believes it is consuming (first and last value against global memory, bit for bit): a refill that
// overtakes a reader, or a wait on the wrong mbarrier phase, changes them.
#ifdef RBG_CHECKED
#define RBG_CHECK_STAGE(fs, src, n)                                                                                        \
    do {                                                                                                                     \
        if ((threadIdx.x & 31) == 0)                                                                                         \
            RBG_CHECK(__double_as_longlong((fs)[0]) == __double_as_longlong(__ldg(src)) &&                                   \
                      __double_as_longlong((fs)[(n) - 1]) == __double_as_longlong(__ldg((src) + (n) - 1)), CHK_STAGE_CONTENT); \
    } while (0)
#else
#define RBG_CHECK_STAGE(fs, src, n) ((void)0)
#endif

// Momentum of a cell centre exactly as the host tables (1/E_p, v = p / E_p: rbg.cu) and the oracle compute it,
// pmin + (i + 1/2) delta in two roundings (this file is compiled with -fmad=false).  A fused form differs by an ulp, which
// is harmless everywhere except at a centre that is zero up to rounding: there a massless species has E_p ~ 1e-16 and
// v = p / E_p depends on that ulp, so the kernels must use the very p that went into the tables.
__device__ __forceinline__ double cell_centre(int i, double delta, double pmin) { return pmin + ((double)i + 0.5) * delta; }

enum { N_MOMENTS = 14 };   // n, jx, jy, jz, T00, T01, T02, T03, T11, T12, T13, T22, T23, T33

struct SpeciesTables {
    const double* iE;        // 1 / E_p per momentum cell (0 where E_p = 0)
    const double* v;         // velocities p / E_p: [3][np]
    double pmin[3], delta[3];
    int n[3];
    int np;
    double mass, charge;
};

// ---------------------------------------------------------------------------------------------------------------
// Moments.  Momentum integrals are midpoint sums, Int d3p -> Sum dp^3.
// With g = f / E and q = |p|^2 + m^2 (so E f = q g):
//   n = S f, T^{0k} = S p_k f, j^k = S p_k g, T^{ik} = S p_i p_k g, T^{00} = S q g.
// A lane owns columns of fixed (ipy, ipz) and walks along ipx, so that only five running sums need the per-cell
// arithmetic (X0 = S_x f, X1 = S_x px f, G0 = S_x g, G1 = S_x px g, G2 = S_x px^2 g); the p_y, p_z factors are applied
// once per column.  Loads are coalesced across the lanes of a warp (consecutive (ipy, ipz)).
// ---------------------------------------------------------------------------------------------------------------
// Persistent kernel, one CTA of 512 threads per SM.  Shared memory holds the species' 1/E table (read for every spatial
// cell) and a ring of stages; a stage is a group of consecutive spatial cells of f (contiguous in memory), filled by one
// TMA bulk copy that completes on the stage's mbarrier while earlier stages are being reduced, so the bytes in flight
// are set by the ring (64 KB and more per SM), not by registers or occupancy.  A group whose byte count or address is
// not a multiple of 16 (an odd leading cell, the tail of the domain) is copied cooperatively with plain loads instead.
// The cells of a stage are shared out among teams of `team` threads (a power of two, 32..512: about one thread per
// (ipy, ipz) column), so small momentum grids keep every warp busy.
enum { MOM_MAX_STAGES = 8, MOM_THREADS = 512, MOM_RED = 4 };   // MOM_RED: reduction buffers ([16 warps][16] doubles each)

// Sum of v[m] over the 32 lanes for 16 values at once: each step halves the number of values a lane carries, so the
// whole reduction takes 8 + 4 + 2 + 1 + 1 shuffles instead of 16 x 5.  On return lane l (l < 16) holds the total of
// value index rev4(l) (bit-reversed), see mom_slot().
__device__ __forceinline__ double warp_reduce16(double (&v)[16], int lane) {
#pragma unroll
    for (int half = 8, bit = 1; half >= 1; half >>= 1, bit <<= 1) {
        const bool up = (lane & bit) != 0;
#pragma unroll
        for (int k = 0; k < half; ++k) {
            const double send = up ? v[k] : v[k + half];
            const double keep = up ? v[k + half] : v[k];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
        }
    }
    return v[0] + __shfl_xor_sync(0xffffffffu, v[0], 16);
}
// value index held by lane l after warp_reduce16: bit j of l selects the upper half at step j
__device__ __forceinline__ int mom_slot(int l) { return ((l & 1) << 3) | ((l & 2) << 1) | ((l & 4) >> 1) | ((l & 8) >> 3); }

// MOM_MAXC = columns a thread owns at a time (1 when the team covers the (ipy, ipz) plane)
// IE_SMEM: the 1/E table is copied to shared memory; when it does not fit next to two stages it is read through L1.
// ONE_TEAM (the whole CTA works on one spatial cell at a time: large momentum grids): no CTA barrier in the steady state.
// Each warp leaves its 14 partial sums in shared memory and bumps a counter; the warp that arrives last adds the 16
// partials in a fixed order and writes the result, and the warp that finishes last with a stage refills it, so warps
// that are done (or own no columns) run ahead to the next stage instead of waiting.
template <int MOM_MAXC, bool IE_SMEM, bool ONE_TEAM>
__global__ void __launch_bounds__(MOM_THREADS, 1)
moments_kernel(const double* __restrict__ f_species, SpeciesTables tb, int nx_cells, double* __restrict__ M_species,
               int group, int n_stages, int team, int lead) {
    extern __shared__ __align__(128) unsigned char mom_smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(mom_smem);                             // MOM_MAX_STAGES mbarriers
    int* done = reinterpret_cast<int*>(mom_smem + 64);                                  // [8] warps done with stage k
    int* cnt = done + MOM_MAX_STAGES;                                                   // [MOM_RED] warps done with a cell
    // reduction buffers: ONE_TEAM one per (stage, cell of the stage) (n_stages * group <= MOM_RED), else two (alternating)
    double* red = reinterpret_cast<double*>(mom_smem + 128);
    double* px_tab = red + (size_t)MOM_RED * (MOM_THREADS / 32) * 16;                   // p_x of the n[0] cell centres
    const size_t head = (128 + ((size_t)MOM_RED * (MOM_THREADS / 32) * 16 + (size_t)tb.n[0]) * 8 + 127) & ~(size_t)127;
    const size_t np = (size_t)tb.np;
    const size_t tab_bytes = IE_SMEM ? (np * 8 + 127) & ~(size_t)127 : 0;
    const double* __restrict__ iEs = IE_SMEM ? reinterpret_cast<const double*>(mom_smem + head) : tb.iE;
    const size_t stage_bytes = ((size_t)group * np * 8 + 127) & ~(size_t)127;
    unsigned char* ring = mom_smem + head + tab_bytes;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nyz = tb.n[1] * tb.n[2];
    // units: [0, lead) (if lead > 0), then groups of `group` cells
    const int n_units = (lead ? 1 : 0) + (nx_cells - lead + group - 1) / group;
    auto unit_first = [&](int u) { return lead ? (u == 0 ? 0 : lead + (u - 1) * group) : u * group; };
    auto unit_cells = [&](int u) { return (lead && u == 0) ? lead : min(group, nx_cells - unit_first(u)); };
    auto unit_tma = [&](int u) {
        return ((size_t)unit_cells(u) * np * 8) % 16 == 0 && reinterpret_cast<uintptr_t>(f_species + (size_t)unit_first(u) * np) % 16 == 0;
    };
    auto arm = [&](int slot, int u) {
        if (u < n_units && unit_tma(u)) {
            const uint32_t bytes = (uint32_t)((size_t)unit_cells(u) * np * 8);
            mbar_expect_tx(&bars[slot], bytes);
            tma_bulk_g2s(ring + (size_t)slot * stage_bytes, f_species + (size_t)unit_first(u) * np, bytes, &bars[slot]);
        }
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < n_stages; ++k) { mbar_init(&bars[k], 1); done[k] = 0; }
        for (int k = 0; k < MOM_RED; ++k) cnt[k] = 0;
        fence_mbar_init();
        for (int k = 0; k < n_stages; ++k) arm(k, blockIdx.x + k * gridDim.x);          // prologue: fill the ring
    }
    for (int i = threadIdx.x; i < tb.n[0]; i += MOM_THREADS) px_tab[i] = cell_centre(i, tb.delta[0], tb.pmin[0]);
    if (IE_SMEM) {
        double* dst = reinterpret_cast<double*>(mom_smem + head);
        for (size_t j = threadIdx.x; j < np; j += MOM_THREADS) dst[j] = __ldg(tb.iE + j);
    }
    __syncthreads();
    const double msq = tb.mass * tb.mass;
    const double dp3 = tb.delta[0] * tb.delta[1] * tb.delta[2];
    const int n_teams = MOM_THREADS / team, my_team = threadIdx.x / team, t_in_team = threadIdx.x - my_team * team;
    const int warps_per_team = team >> 5, warp_in_team = t_in_team >> 5;
    int it = 0, flip = 0;
    uint32_t phases = 0;                                       // bit k: parity of the next completion of stage k
    for (int u = blockIdx.x; u < n_units; u += gridDim.x, ++it) {
        const int slot = it % n_stages;
        double* fs = reinterpret_cast<double*>(ring + (size_t)slot * stage_bytes);
        const int cells = unit_cells(u), first = unit_first(u);
        if (unit_tma(u)) {
            mbar_wait(&bars[slot], (phases >> slot) & 1u);
            phases ^= 1u << slot;
        } else {
            if (ONE_TEAM) __syncthreads();                     // nobody still reads the unit this slot held before
            const double* src = f_species + (size_t)first * np;
            for (size_t j = threadIdx.x; j < (size_t)cells * np; j += MOM_THREADS) fs[j] = __ldcs(src + j);
            __syncthreads();
        }
        RBG_CHECK_STAGE(fs, f_species + (size_t)first * np, (size_t)cells * np);
        RBG_CHECK(first + cells <= nx_cells && (size_t)(slot + 1) * stage_bytes + head + tab_bytes <= dynamic_smem_size(), CHK_BE_INDEX);
        for (int cell0 = 0; cell0 < cells; cell0 += n_teams) {           // one round: every team reduces one cell
            const int cell = cell0 + my_team;
            const bool active = cell < cells;
            const double* __restrict__ fc = fs + (size_t)(active ? cell : 0) * np;
            double acc[16];
#pragma unroll
            for (int m = 0; m < 16; ++m) acc[m] = 0.0;
            // a thread owns columns c = t_in_team + q * team of fixed (ipy, ipz) and walks along ipx
            for (int c0 = t_in_team; active && c0 - lane < nyz; c0 += team * MOM_MAXC) {
                double X0[MOM_MAXC], X1[MOM_MAXC], G0[MOM_MAXC], G1[MOM_MAXC], G2[MOM_MAXC];
#pragma unroll
                for (int q = 0; q < MOM_MAXC; ++q) { X0[q] = X1[q] = G0[q] = G1[q] = G2[q] = 0.0; }
#pragma unroll
                for (int q = 0; q < MOM_MAXC; ++q) {
                    const int c = c0 + q * team;
                    if (c < nyz) {
                        const double* __restrict__ pf = fc + c;
                        const double* __restrict__ pe = iEs + c;
                        // two independent sets of running sums (even / odd planes) halve the dependent-add chains
                        double x0 = 0.0, x1 = 0.0, g0 = 0.0, g1 = 0.0, g2 = 0.0;
                        double y0 = 0.0, y1 = 0.0, h0 = 0.0, h1 = 0.0, h2 = 0.0;
                        const int n0e = tb.n[0] & ~1;
#pragma unroll 2
                        for (int i = 0; i < n0e; i += 2) {
                            const double pxa = px_tab[i], pxb = px_tab[i + 1];
                            const double a = pf[(size_t)i * nyz], b = pf[(size_t)(i + 1) * nyz];
                            const double ga = a * (IE_SMEM ? pe[(size_t)i * nyz] : __ldg(pe + (size_t)i * nyz));
                            const double gb = b * (IE_SMEM ? pe[(size_t)(i + 1) * nyz] : __ldg(pe + (size_t)(i + 1) * nyz));
                            const double pga = pxa * ga, pgb = pxb * gb;
                            x0 += a;                 y0 += b;
                            x1 = fma(pxa, a, x1);    y1 = fma(pxb, b, y1);
                            g0 += ga;                h0 += gb;
                            g1 += pga;               h1 += pgb;
                            g2 = fma(pxa, pga, g2);  h2 = fma(pxb, pgb, h2);
                        }
                        if (n0e < tb.n[0]) {
                            const int i = n0e;
                            const double px = px_tab[i];
                            const double a = pf[(size_t)i * nyz];
                            const double g = a * (IE_SMEM ? pe[(size_t)i * nyz] : __ldg(pe + (size_t)i * nyz));
                            const double pg = px * g;
                            x0 += a; x1 = fma(px, a, x1); g0 += g; g1 += pg; g2 = fma(px, pg, g2);
                        }
                        x0 += y0; x1 += y1; g0 += h0; g1 += h1; g2 += h2;
                        X0[q] = x0; X1[q] = x1; G0[q] = g0; G1[q] = g1; G2[q] = g2;
                    }
                }
#pragma unroll
                for (int q = 0; q < MOM_MAXC; ++q) {
                    const int c = c0 + q * team;
                    if (c < nyz) {
                        const int iy = c / tb.n[2], iz = c - iy * tb.n[2];
                        const double py = cell_centre(iy, tb.delta[1], tb.pmin[1]);
                        const double pz = cell_centre(iz, tb.delta[2], tb.pmin[2]);
                        const double r = fma(py, py, fma(pz, pz, msq));                   // q - px^2
                        const double yG0 = py * G0[q], zG0 = pz * G0[q];
                        acc[0] += X0[q];                                                  // n
                        acc[1] += G1[q]; acc[2] += yG0; acc[3] += zG0;                    // j
                        acc[4] += fma(r, G0[q], G2[q]);                                   // T00 = S (px^2 + r) g
                        acc[5] += X1[q]; acc[6] = fma(py, X0[q], acc[6]); acc[7] = fma(pz, X0[q], acc[7]);      // T0k
                        acc[8] += G2[q]; acc[9] = fma(py, G1[q], acc[9]); acc[10] = fma(pz, G1[q], acc[10]);    // Txx Txy Txz
                        acc[11] = fma(py, yG0, acc[11]); acc[12] = fma(py, zG0, acc[12]); acc[13] = fma(pz, zG0, acc[13]);
                    }
                }
            }
            const double tot = warp_reduce16(acc, lane);
            if (ONE_TEAM) {
                const int rbi = slot * group + cell;
                double* rb = red + (size_t)rbi * (MOM_THREADS / 32) * 16;
                if (lane < 16) rb[warp * 16 + mom_slot(lane)] = tot;
                __syncwarp();
                int last = 0;
                if (lane == 0) {
                    __threadfence_block();
                    last = atomicAdd(&cnt[rbi], 1) == MOM_THREADS / 32 - 1;
                    if (last) cnt[rbi] = 0;
                }
                last = __shfl_sync(0xffffffffu, last, 0);
                if (last) {                                    // every warp's partial sums are in rb
                    __threadfence_block();
                    if (lane < N_MOMENTS) {
                        double v = 0.0;
#pragma unroll
                        for (int w = 0; w < MOM_THREADS / 32; ++w) v += rb[w * 16 + lane];
                        M_species[((size_t)first + cell) * N_MOMENTS + lane] = v * dp3;
                    }
                }
            } else {
                double* rb = red + (size_t)flip * (MOM_THREADS / 32) * 16;
                if (lane < 16) rb[warp * 16 + mom_slot(lane)] = tot;
                __syncthreads();
                if (active && t_in_team < N_MOMENTS) {
                    double v = 0.0;
                    for (int w = 0; w < warps_per_team; ++w) v += rb[(my_team * warps_per_team + w) * 16 + t_in_team];
                    M_species[((size_t)first + cell) * N_MOMENTS + t_in_team] = v * dp3;
                }
                flip ^= 1;                                     // the next round writes the other buffer: one barrier per round
            }
        }
        RBG_CHECK_STAGE(fs, f_species + (size_t)first * np, (size_t)cells * np);
        if (ONE_TEAM) {
            // the warp that finishes last with this stage refills it (its reads of the stage and of the reduction
            // buffers are complete: their values were consumed above)
            __syncwarp();
            if (lane == 0) {
                __threadfence_block();
                if (atomicAdd(&done[slot], 1) == MOM_THREADS / 32 - 1) {
                    done[slot] = 0;
                    arm(slot, u + n_stages * gridDim.x);
                }
            }
        } else {
            __syncthreads();                                   // every team has finished reading the stage
            if (threadIdx.x == 0) arm(slot, u + n_stages * gridDim.x);   // refill with the unit n_stages iterations ahead
        }
    }
    (void)warp_in_team;
}

// ---------------------------------------------------------------------------------------------------------------
// Moments on a momentum grid that is symmetric about p = 0 in all three directions (every workload of the paper), one
// spatial cell per stage.  Same sums as moments_kernel; what the symmetry buys:
//   * 1/E_p depends on |p_x|, |p_y|, |p_z| only, so its table shrinks to one octant (8 KB instead of 64 KB at 20^3) and the
//     ring gets a third stage;
//   * the planes +p_x and -p_x of a column share 1/E: with s = a_+ + a_-, d = a_+ - a_- the five running sums of a column
//     take X0 += s, X1 += p_x d, G0 += e s, G1 += p_x (e d), G2 += p_x^2 (e s): 9 FP64 instructions per pair of cells
//     instead of 14, 3 shared-memory loads instead of 6;
//   * a thread always owns the same (at most MS_MAXC) columns, so p_y, p_z, p_y^2 + p_z^2 + m^2 and the table offset
//     are computed once per kernel, not once per cell.
// The CTA is two teams of 8 warps; a team takes every other unit of the CTA, so two cells are reduced at a time (each
// lane carries up to two columns: the 16-value butterfly and the cross-warp sum are paid by 8 warps per cell instead
// of 16) while the third stage is in flight.  No CTA barrier after the prologue: the last warp of a team to finish a
// stage re-arms it (mbarrier + bulk copy) for the unit three further on, which the other team will consume.
// ---------------------------------------------------------------------------------------------------------------
enum { MS_THREADS = 512, MS_TEAM = 256, MS_STAGES = 3, MS_MAXC = 2 };

__global__ void __launch_bounds__(MS_THREADS, 1)
moments_sym_kernel(const double* __restrict__ f_species, SpeciesTables tb, int nx_cells, double* __restrict__ M_species) {
    extern __shared__ __align__(128) unsigned char mom_smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(mom_smem);                             // 2 MS_STAGES mbarriers: [slot][fill & 1]
    int* done = reinterpret_cast<int*>(mom_smem + 64);                                  // [MS_STAGES] warps done with the stage
    int* cnt = done + MS_STAGES;                                                        // [MS_STAGES] warps whose partial sums are in
    double* red = reinterpret_cast<double*>(mom_smem + 128);                            // [MS_STAGES][8 warps][16]
    const int c0 = tb.n[0] >> 1, odd0 = tb.n[0] & 1, c1 = tb.n[1] >> 1, odd1 = tb.n[1] & 1, c2 = tb.n[2] >> 1, odd2 = tb.n[2] & 1;
    const int n0h = c0 + odd0, n1h = c1 + odd1, n2h = c2 + odd2, nyzh = n1h * n2h;
    double* pxs = red + MS_STAGES * (MS_TEAM / 32) * 16;                                // [c0] p_x of the planes above the centre
    double* px2s = pxs + c0;                                                            // [c0] their squares
    double* iEc = px2s + c0;                                                            // [n0h][n1h][n2h] 1/E of one octant
    const size_t np = (size_t)tb.np;
    const size_t head = (128 + ((size_t)MS_STAGES * (MS_TEAM / 32) * 16 + 2 * (size_t)c0 + (size_t)n0h * nyzh) * 8 + 127) & ~(size_t)127;
    const size_t stage_bytes = (np * 8 + 127) & ~(size_t)127;
    unsigned char* ring = mom_smem + head;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int team = warp >> 3, wt = warp & 7;                                          // team 0 / 1, warp within the team
    const int nyz = tb.n[1] * tb.n[2];
    const int n_units = (nx_cells - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // units k = 0.. of this CTA: cell blockIdx.x + k gridDim.x
    // Fill number m = k / 3 of slot k % 3 completes on mbarrier [slot][m & 1].  The fills of a slot alternate between the
    // teams, so each barrier belongs to one team: its previous fill (m - 2) was waited on by the same team and its next one
    // (m + 2) cannot be armed before that team has consumed fill m -- the barrier is either in phase m >> 1 (in flight) or
    // one past it (landed), which the parity wait tells apart.  (One barrier per slot would not do: a team about to wait for
    // fill m could find it in phase m - 1, m or m + 1.)
    auto arm = [&](int slot, int k) {
        if (k < n_units) {
            uint64_t* bar = &bars[2 * slot + ((k / MS_STAGES) & 1)];
            mbar_expect_tx(bar, (uint32_t)(np * 8));
            tma_bulk_g2s(ring + (size_t)slot * stage_bytes, f_species + ((size_t)blockIdx.x + (size_t)k * gridDim.x) * np, (uint32_t)(np * 8), bar);
        }
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < MS_STAGES; ++k) { mbar_init(&bars[2 * k], 1); mbar_init(&bars[2 * k + 1], 1); done[k] = 0; cnt[k] = 0; }
        fence_mbar_init();
        for (int k = 0; k < MS_STAGES; ++k) arm(k, k);
    }
    // rows 0 .. c0-1 of the octant table: the planes above the centre (pair j = planes c0 + odd0 + j and c0 - 1 - j);
    // row c0 (odd n only): the centre plane p_x = 0.  Likewise in y and z.
    for (int i = threadIdx.x; i < c0; i += MS_THREADS) {
        const double px = cell_centre((c0 + odd0 + i), tb.delta[0], tb.pmin[0]);
        pxs[i] = px; px2s[i] = px * px;
    }
    for (int i = threadIdx.x; i < n0h * nyzh; i += MS_THREADS) {
        const int j0 = i / nyzh, r = i - j0 * nyzh, j1 = r / n2h, j2 = r - j1 * n2h;
        const int i0 = j0 < c0 ? c0 + odd0 + j0 : c0, i1 = j1 < c1 ? c1 + odd1 + j1 : c1, i2 = j2 < c2 ? c2 + odd2 + j2 : c2;
        iEc[i] = __ldg(tb.iE + ((size_t)i0 * tb.n[1] + i1) * tb.n[2] + i2);
    }
    // this thread's columns (fixed for the whole kernel) and everything that depends on the column only
    int col[MS_MAXC], cm[MS_MAXC];
    bool valid[MS_MAXC];
    double py[MS_MAXC], pz[MS_MAXC], rr[MS_MAXC];
    const double msq = tb.mass * tb.mass;
#pragma unroll
    for (int q = 0; q < MS_MAXC; ++q) {
        const int c = wt * 32 + lane + q * MS_TEAM;
        valid[q] = c < nyz;
        col[q] = valid[q] ? c : nyz - 1;                                  // an idle slot reads a valid column and is discarded
        const int iy = col[q] / tb.n[2], iz = col[q] - iy * tb.n[2];
        py[q] = cell_centre(iy, tb.delta[1], tb.pmin[1]);
        pz[q] = cell_centre(iz, tb.delta[2], tb.pmin[2]);
        rr[q] = fma(py[q], py[q], fma(pz[q], pz[q], msq));               // E^2 - p_x^2
        const int m1 = iy >= c1 + odd1 ? iy - c1 - odd1 : (iy < c1 ? c1 - 1 - iy : c1);
        const int m2 = iz >= c2 + odd2 ? iz - c2 - odd2 : (iz < c2 ? c2 - 1 - iz : c2);
        cm[q] = m1 * n2h + m2;
    }
    const bool second = __any_sync(0xffffffffu, valid[1]);               // warp-uniform: does any lane carry a second column
    const double dp3 = tb.delta[0] * tb.delta[1] * tb.delta[2];
    __syncthreads();
    for (int k = team; k < n_units; k += 2) {
        const int slot = k % MS_STAGES;
        const size_t cell = (size_t)blockIdx.x + (size_t)k * gridDim.x;
        const double* __restrict__ fc = reinterpret_cast<const double*>(ring + (size_t)slot * stage_bytes);
        mbar_wait(&bars[2 * slot + ((k / MS_STAGES) & 1)], (uint32_t)(k / (2 * MS_STAGES)) & 1u);
        RBG_CHECK_STAGE(fc, f_species + cell * np, np);
        RBG_CHECK(cell < (size_t)nx_cells && (size_t)(slot + 1) * stage_bytes + head <= dynamic_smem_size(), CHK_BE_INDEX);
        double acc[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) acc[m] = 0.0;
#pragma unroll
        for (int q = 0; q < MS_MAXC; ++q) {
            if (q == 1 && !second) break;
            const double* __restrict__ pf = fc + col[q];
            const double* __restrict__ pe = iEc + cm[q];
            double x0 = 0.0, x1 = 0.0, g0 = 0.0, g1 = 0.0, g2 = 0.0;
            if (odd0) {                                                  // centre plane: p_x = 0
                const double a = pf[(size_t)c0 * nyz];
                x0 = a; g0 = a * pe[(size_t)c0 * nyzh];
            }
#pragma unroll 5
            for (int j = 0; j < c0; ++j) {
                const double ap = pf[(size_t)(c0 + odd0 + j) * nyz], am = pf[(size_t)(c0 - 1 - j) * nyz];
                const double e = pe[(size_t)j * nyzh], px = pxs[j], px2 = px2s[j];
                const double sm = ap + am, df = ap - am;
                const double es = e * sm, ed = e * df;
                x0 += sm;
                x1 = fma(px, df, x1);
                g0 += es;
                g1 = fma(px, ed, g1);
                g2 = fma(px2, es, g2);
            }
            if (!valid[q]) { x0 = x1 = g0 = g1 = g2 = 0.0; }
            const double yG0 = py[q] * g0, zG0 = pz[q] * g0;
            acc[0] += x0;                                                                     // n
            acc[1] += g1; acc[2] += yG0; acc[3] += zG0;                                       // j
            acc[4] += fma(rr[q], g0, g2);                                                     // T00 = S (px^2 + r) g
            acc[5] += x1; acc[6] = fma(py[q], x0, acc[6]); acc[7] = fma(pz[q], x0, acc[7]);   // T0k
            acc[8] += g2; acc[9] = fma(py[q], g1, acc[9]); acc[10] = fma(pz[q], g1, acc[10]); // Txx Txy Txz
            acc[11] = fma(py[q], yG0, acc[11]); acc[12] = fma(py[q], zG0, acc[12]); acc[13] = fma(pz[q], zG0, acc[13]);
        }
        RBG_CHECK_STAGE(fc, f_species + cell * np, np);
        const double tot = warp_reduce16(acc, lane);
        double* rb = red + (size_t)slot * (MS_TEAM / 32) * 16;
        if (lane < 16) rb[wt * 16 + mom_slot(lane)] = tot;
        __syncwarp();
        int last = 0;
        if (lane == 0) {
            __threadfence_block();
            last = atomicAdd(&cnt[slot], 1) == MS_TEAM / 32 - 1;
            if (last) cnt[slot] = 0;
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last) {                                                      // the partial sums of all 8 warps of the team are in rb
            __threadfence_block();
            if (lane < N_MOMENTS) {
                double v = 0.0;
#pragma unroll
                for (int w = 0; w < MS_TEAM / 32; ++w) v += rb[w * 16 + lane];
                M_species[cell * N_MOMENTS + lane] = v * dp3;
            }
        }
        // the warp that finishes last with this stage (its reads of the stage and of rb are complete) refills it
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            if (atomicAdd(&done[slot], 1) == MS_TEAM / 32 - 1) {
                done[slot] = 0;
                arm(slot, k + MS_STAGES);
            }
        }
    }
}

// total[ix][m] = Sum_a M[a][ix][m] (Eq. 7, 9); em[ix][0..3] = Sum_a Q_a (n_a, j_a) (Eq. 15).  Either may be null.
__global__ void totals_kernel(const double* __restrict__ M, const double* __restrict__ charges, int n_species, int nx_cells,
                              double* __restrict__ total, double* __restrict__ em) {
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i >= (size_t)nx_cells * N_MOMENTS) return;
    const int m = (int)(i % N_MOMENTS);
    const size_t ix = i / N_MOMENTS;
    double t = 0.0, q = 0.0;
    for (int s = 0; s < n_species; ++s) {
        const double v = M[((size_t)s * nx_cells + ix) * N_MOMENTS + m];
        t += v;
        q = fma(charges[s], v, q);
    }
    if (total) total[i] = t;
    if (em && m < 4) em[ix * 4 + m] = q;
}

// ---------------------------------------------------------------------------------------------------------------
// UPFD stencils.  Both steps have the form (reading R23)
//     f_new = [ f/3 + Sum_d c_d f_up,d ] / [ 1/3 + Sum_d c_d ],
// with c_d = dt |v_d| / dx_d and f_up,d the spatial neighbour on the upwind side (drift, Eq. 30), or
// c_d = dt |F_d| / dp_d and the momentum neighbour on the upwind side of the force (Vlasov, Eq. 34).
// A thread owns one momentum cell (its velocity stays in registers) and walks over a slab of consecutive spatial
// cells; a warp reads and writes 256 contiguous bytes per spatial cell.
// ---------------------------------------------------------------------------------------------------------------
struct DriftParams {
    double dt;
    double inv_dx[3];
    int nxyz[3];
    int bc[3];               // 1 periodic, 0 wall with reflection probability zeta
    double zeta;
    int zseg;                // cells of a z row per CTA
    int tile_y;              // rows per y tile (CTA order: y tile, i_x, row in tile, z segment, momentum chunk)
};

enum { STENCIL_BATCH = 4 };  // spatial cells whose loads are issued together (measured on config 4: 3, 6, 8 are slower)

// CTA = (momentum chunk of 256 cells) x (segment of a z row).  CTAs are ordered so that consecutive CTAs walk along x
// inside a tile of tile_y rows: the x neighbour of a cell was read tile_y * nz spatial cells earlier and is still in
// L2 (for a 32^3 x 20^3 grid a whole x plane is 65 MB away in memory order, which L2 does not hold next to the output).
__global__ void __launch_bounds__(256, 4)
drift_upfd_kernel(const double* __restrict__ f_species, double* __restrict__ out_species, SpeciesTables tb, DriftParams dp) {
    const int nchunks = (tb.np + blockDim.x - 1) / blockDim.x;
    const int nzseg = (dp.nxyz[2] + dp.zseg - 1) / dp.zseg;
    int b = blockIdx.x;
    const int chunk = b % nchunks; b /= nchunks;
    const int zs = b % nzseg; b /= nzseg;
    const int iy_in = b % dp.tile_y; b /= dp.tile_y;
    const int ixx = b % dp.nxyz[0];
    const int iy = (b / dp.nxyz[0]) * dp.tile_y + iy_in;
    const int ip = chunk * blockDim.x + threadIdx.x;
    if (ip >= tb.np || iy >= dp.nxyz[1]) return;
    const int z0 = zs * dp.zseg, z1 = min(z0 + dp.zseg, dp.nxyz[2]);
    const ptrdiff_t np = tb.np;
    // per-momentum-cell constants
    double c[3];
    int sgn[3], mir[3];
    {
        const int nyz = tb.n[1] * tb.n[2];
        const int i0 = ip / nyz, i1 = (ip - i0 * nyz) / tb.n[2], i2 = ip - i0 * nyz - i1 * tb.n[2];
        mir[0] = ip + (tb.n[0] - 1 - 2 * i0) * nyz;      // momentum cell with p_d reversed (grids symmetric about 0)
        mir[1] = ip + (tb.n[1] - 1 - 2 * i1) * tb.n[2];
        mir[2] = ip + (tb.n[2] - 1 - 2 * i2);
    }
    double den = 1.0 / 3.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double v = __ldg(tb.v + (size_t)d * tb.np + ip);
        c[d] = (dp.dt * fabs(v)) * dp.inv_dx[d];
        sgn[d] = v > 0.0 ? 1 : -1;
        den += c[d];
    }
    const double rden = 1.0 / den;
    // upwind neighbour along d of the spatial cell with index i along d: an interior or periodic neighbour (offset in
    // spatial cells, weight c_d) or the wall ghost zeta * f(same cell, mirrored momentum)
    const int stride[3] = {dp.nxyz[1] * dp.nxyz[2], dp.nxyz[2], 1};
    auto upwind = [&](int d, int i, ptrdiff_t& off, double& cs) {
        const int j = i - sgn[d];
        const bool inside = (unsigned)j < (unsigned)dp.nxyz[d];
        const bool real = inside || dp.bc[d] == 1;
        const int jn = inside ? j : (j < 0 ? dp.nxyz[d] - 1 : 0);
        off = real ? (ptrdiff_t)((jn - i) * stride[d]) * np + ip : (ptrdiff_t)mir[d];
        cs = real ? c[d] : c[d] * dp.zeta;
    };
    ptrdiff_t offx, offy;
    double csx, csy;
    upwind(0, ixx, offx, csx);
    upwind(1, iy, offy, csy);
    const size_t row0 = ((size_t)ixx * dp.nxyz[1] + iy) * dp.nxyz[2];
    // Walk the z segment in the direction of v_z, so that the upwind z neighbour of a cell is the cell visited just before
    // it: three loads per cell (itself, the x and the y neighbour) instead of four, and only the first cell of the walk needs
    // the general neighbour rule (interior / periodic / wall ghost).  Lanes with v_z < 0 walk down while the others walk up;
    // each still reads and writes runs of consecutive momentum cells.
    const int len = z1 - z0, zstart = sgn[2] > 0 ? z0 : z1 - 1;
    const ptrdiff_t step = sgn[2] > 0 ? np : -np;
    const double* __restrict__ ps = f_species + (row0 + zstart) * np;            // momentum block of the cell being visited
    double* __restrict__ po = out_species + (row0 + zstart) * np + ip;
    ptrdiff_t offz;
    double cz;
    upwind(2, zstart, offz, cz);
#ifdef RBG_CHECKED
    const ptrdiff_t total = (ptrdiff_t)dp.nxyz[0] * dp.nxyz[1] * dp.nxyz[2] * np;
    {
        const ptrdiff_t base = (ptrdiff_t)(row0 + zstart) * np;
        RBG_CHECK(base + offz >= 0 && base + offz < total, CHK_BE_INDEX);
    }
#endif
    double prev = __ldg(ps + offz);                                             // upwind z neighbour (or wall ghost) of the first cell
    const double third = 1.0 / 3.0;
    for (int t = 0; t < len; t += STENCIL_BATCH) {
        double self[STENCIL_BATCH], ux[STENCIL_BATCH], uy[STENCIL_BATCH];
#pragma unroll
        for (int k = 0; k < STENCIL_BATCH; ++k) {
            const double* __restrict__ row = ps + (ptrdiff_t)min(k, len - 1 - t) * step;    // the tail repeats the last cell (not stored)
#ifdef RBG_CHECKED
            {   // every address of the stencil lies inside the species block
                const ptrdiff_t base = row - f_species;
                RBG_CHECK(base + ip >= 0 && base + ip < total && base + offx >= 0 && base + offx < total && base + offy >= 0 &&
                          base + offy < total, CHK_BE_INDEX);
            }
#endif
            self[k] = __ldg(row + ip);
            ux[k] = __ldg(row + offx);
            uy[k] = __ldg(row + offy);
        }
#pragma unroll
        for (int k = 0; k < STENCIL_BATCH; ++k) {
            if (t + k < len) {
                const double num = fma(cz, prev, fma(csy, uy[k], fma(csx, ux[k], self[k] * third)));
                __stcs(po + (ptrdiff_t)k * step, num * rden);
                prev = self[k];
                cz = c[2];                                                       // every later cell has an interior neighbour
            }
        }
        ps += (ptrdiff_t)STENCIL_BATCH * step;
        po += (ptrdiff_t)STENCIL_BATCH * step;
    }
}

// Second-order positivity-preserving flux-limited drift step, Eq. 31-33, periodic.  Face value
// between the upwind cell c and the downwind cell r, l being the cell upwind of c (reading R26):
//   fc + 1/2 phi (fc - fl),  phi = max(0, min(1, (fr - fc)/(fc - fl), 2 / max(theta, (fl - fc)/fc))).
// Division-free form of the same value: with a = fr - fc and d = fc - fl, phi d = 0 when a d <= 0 (r <= 0); otherwise
// min(1, r) d = (|a| < |d| ? a : d), and the positivity limiter 2 fc / (fl - fc) (binding only for fl > fc, i.e. d < 0,
// where 2/theta never is) caps |phi d| at 2 fc.
__device__ __forceinline__ double limited_face(double fl, double fc, double fr) {
    const double d = fc - fl, a = fr - fc;
    double t = fabs(a) < fabs(d) ? a : d;
    if (d < 0.0) t = fmax(t, -2.0 * fc);
    if (!(a * d > 0.0) || fc == 0.0) t = 0.0;
    return fma(0.5, t, fc);
}

// Same decomposition and CTA order as drift_upfd_kernel.  f(t+dt) = f - 3 dt Sum_d |v_d| (O_d - I_d) / dx_d with O the face
// value leaving the cell and I the one entering it.
__global__ void __launch_bounds__(256)
drift_pfl_kernel(const double* __restrict__ f_species, double* __restrict__ out_species, SpeciesTables tb, DriftParams dp) {
    const int nchunks = (tb.np + blockDim.x - 1) / blockDim.x;
    const int nzseg = (dp.nxyz[2] + dp.zseg - 1) / dp.zseg;
    int b = blockIdx.x;
    const int chunk = b % nchunks; b /= nchunks;
    const int zs = b % nzseg; b /= nzseg;
    const int iy_in = b % dp.tile_y; b /= dp.tile_y;
    const int ixx = b % dp.nxyz[0];
    const int iy = (b / dp.nxyz[0]) * dp.tile_y + iy_in;
    const int ip = chunk * blockDim.x + threadIdx.x;
    if (ip >= tb.np || iy >= dp.nxyz[1]) return;
    const int z0 = zs * dp.zseg, z1 = min(z0 + dp.zseg, dp.nxyz[2]);
    const ptrdiff_t np = tb.np;
    double c[3];
    int sgn[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double v = __ldg(tb.v + (size_t)d * tb.np + ip);
        c[d] = (3.0 * dp.dt * fabs(v)) * dp.inv_dx[d];
        sgn[d] = v > 0.0 ? 1 : -1;
    }
    const int stride[3] = {dp.nxyz[1] * dp.nxyz[2], dp.nxyz[2], 1};
    // periodic offset (in spatial cells) from index i along d to index i + k
    auto wrap = [&](int d, int i, int k) {                      // |k| <= 2; extents of 1 or 2 wrap more than once
        const int n = dp.nxyz[d];
        int j = i + k;
        j = j < 0 ? j + n : j; j = j < 0 ? j + n : j;
        j = j >= n ? j - n : j; j = j >= n ? j - n : j;
        return (ptrdiff_t)((j - i) * stride[d]) * np;
    };
    ptrdiff_t ox[3], oy[3];                                   // upwind-2, upwind-1, downwind along x and y
    ox[0] = wrap(0, ixx, -2 * sgn[0]); ox[1] = wrap(0, ixx, -sgn[0]); ox[2] = wrap(0, ixx, sgn[0]);
    oy[0] = wrap(1, iy, -2 * sgn[1]);  oy[1] = wrap(1, iy, -sgn[1]);  oy[2] = wrap(1, iy, sgn[1]);
    const size_t row0 = ((size_t)ixx * dp.nxyz[1] + iy) * dp.nxyz[2];
    constexpr int PB = 2;                                     // cells whose ten loads are issued together
    for (int zb = z0; zb < z1; zb += PB) {
        double fc[PB], x2[PB], x1[PB], xd[PB], y2[PB], y1[PB], yd[PB], w2[PB], w1[PB], wd[PB];
#pragma unroll
        for (int k = 0; k < PB; ++k) {
            const int z = min(zb + k, z1 - 1);                       // the tail repeats the last cell (not stored)
            const double* __restrict__ row = f_species + (row0 + z) * np + ip;
            fc[k] = __ldg(row);
            x2[k] = __ldg(row + ox[0]); x1[k] = __ldg(row + ox[1]); xd[k] = __ldg(row + ox[2]);
            y2[k] = __ldg(row + oy[0]); y1[k] = __ldg(row + oy[1]); yd[k] = __ldg(row + oy[2]);
            w2[k] = __ldg(row + wrap(2, z, -2 * sgn[2])); w1[k] = __ldg(row + wrap(2, z, -sgn[2])); wd[k] = __ldg(row + wrap(2, z, sgn[2]));
        }
#pragma unroll
        for (int k = 0; k < PB; ++k) {
            if (zb + k < z1) {
                double div = c[0] * (limited_face(x1[k], fc[k], xd[k]) - limited_face(x2[k], x1[k], fc[k]));
                div = fma(c[1], limited_face(y1[k], fc[k], yd[k]) - limited_face(y2[k], y1[k], fc[k]), div);
                div = fma(c[2], limited_face(w1[k], fc[k], wd[k]) - limited_face(w2[k], w1[k], fc[k]), div);
                __stcs(out_species + (row0 + zb + k) * np + ip, fc[k] - div);
            }
        }
    }
}

struct VlasovParams {
    double dt;
    int nx_cells;
    const double* E;         // [nx_cells][3]
    const double* B;         // [nx_cells][3]
};

// Vlasov step: the stencil lives inside the momentum block of one (species, spatial cell), so the block is staged in
// shared memory exactly like in moments_kernel (persistent CTA, ring of TMA stages, 1/E table resident) and every
// neighbour comes from shared memory: HBM sees f once in and f_out once out.  A thread owns (ipy, ipz) columns and walks
// along ipx; v = p / E_p is rebuilt from the cell centre and the 1/E table; stores are coalesced across the lanes.
template <int VL_MAXC>
__global__ void __launch_bounds__(MOM_THREADS, 1)
vlasov_upfd_kernel(const double* __restrict__ f_species, double* __restrict__ out_species, SpeciesTables tb, VlasovParams vp,
                   int group, int n_stages, int team, int lead) {
    extern __shared__ __align__(128) unsigned char mom_smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(mom_smem);
    int* done = reinterpret_cast<int*>(mom_smem + 64);                                  // warps done with stage k
    double* px_tab = reinterpret_cast<double*>(mom_smem + 128);
    const size_t head = (128 + (size_t)tb.n[0] * 8 + 127) & ~(size_t)127;
    double* iEs = reinterpret_cast<double*>(mom_smem + head);
    const size_t np = (size_t)tb.np;
    const size_t tab_bytes = (np * 8 + 127) & ~(size_t)127;
    const size_t stage_bytes = ((size_t)group * np * 8 + 127) & ~(size_t)127;
    unsigned char* ring = mom_smem + head + tab_bytes;
    const int lane = threadIdx.x & 31;
    const int nx_cells = vp.nx_cells;
    const int nyz = tb.n[1] * tb.n[2], n0 = tb.n[0], n1 = tb.n[1], n2 = tb.n[2];
    const int n_units = (lead ? 1 : 0) + (nx_cells - lead + group - 1) / group;
    auto unit_first = [&](int u) { return lead ? (u == 0 ? 0 : lead + (u - 1) * group) : u * group; };
    auto unit_cells = [&](int u) { return (lead && u == 0) ? lead : min(group, nx_cells - unit_first(u)); };
    auto unit_tma = [&](int u) {
        return ((size_t)unit_cells(u) * np * 8) % 16 == 0 && reinterpret_cast<uintptr_t>(f_species + (size_t)unit_first(u) * np) % 16 == 0;
    };
    auto arm = [&](int slot, int u) {
        if (u < n_units && unit_tma(u)) {
            const uint32_t bytes = (uint32_t)((size_t)unit_cells(u) * np * 8);
            mbar_expect_tx(&bars[slot], bytes);
            tma_bulk_g2s(ring + (size_t)slot * stage_bytes, f_species + (size_t)unit_first(u) * np, bytes, &bars[slot]);
        }
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < n_stages; ++k) { mbar_init(&bars[k], 1); done[k] = 0; }
        fence_mbar_init();
        for (int k = 0; k < n_stages; ++k) arm(k, blockIdx.x + k * gridDim.x);
    }
    for (int i = threadIdx.x; i < n0; i += MOM_THREADS) px_tab[i] = cell_centre(i, tb.delta[0], tb.pmin[0]);
    for (size_t j = threadIdx.x; j < np; j += MOM_THREADS) iEs[j] = __ldg(tb.iE + j);
    __syncthreads();
    const double k0 = vp.dt / tb.delta[0], k1 = vp.dt / tb.delta[1], k2 = vp.dt / tb.delta[2];
    const double Q = tb.charge;
    const int n_teams = MOM_THREADS / team, my_team = threadIdx.x / team, t_in_team = threadIdx.x - my_team * team;
    int it = 0;
    uint32_t phases = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x, ++it) {
        const int slot = it % n_stages;
        double* fs = reinterpret_cast<double*>(ring + (size_t)slot * stage_bytes);
        const int cells = unit_cells(u), first = unit_first(u);
        if (unit_tma(u)) {
            mbar_wait(&bars[slot], (phases >> slot) & 1u);
            phases ^= 1u << slot;
        } else {
            __syncthreads();                                   // nobody still reads the unit this slot held before
            const double* src = f_species + (size_t)first * np;
            for (size_t j = threadIdx.x; j < (size_t)cells * np; j += MOM_THREADS) fs[j] = __ldcs(src + j);
            __syncthreads();
        }
        RBG_CHECK_STAGE(fs, f_species + (size_t)first * np, (size_t)cells * np);
        RBG_CHECK(first + cells <= vp.nx_cells, CHK_BE_INDEX);
        for (int cell = my_team; cell < cells; cell += n_teams) {
            const double* __restrict__ fc = fs + (size_t)cell * np;
            double* __restrict__ oc = out_species + ((size_t)first + cell) * np;
            const double* __restrict__ Ev = vp.E + ((size_t)first + cell) * 3;
            const double* __restrict__ Bv = vp.B + ((size_t)first + cell) * 3;
            // F = Q (E + v x B) with Q folded into the fields of this spatial cell
            const double QEx = Q * __ldg(Ev), QEy = Q * __ldg(Ev + 1), QEz = Q * __ldg(Ev + 2);
            const double QBx = Q * __ldg(Bv), QBy = Q * __ldg(Bv + 1), QBz = Q * __ldg(Bv + 2);
            for (int c0 = t_in_team; c0 - lane < nyz; c0 += team * VL_MAXC) {
#pragma unroll
                for (int q = 0; q < VL_MAXC; ++q) {
                    const int c = c0 + q * team;
                    if (c < nyz) {
                        const int iy = c / n2, iz = c - iy * n2;
                        const double py = cell_centre(iy, tb.delta[1], tb.pmin[1]);
                        const double pz = cell_centre(iz, tb.delta[2], tb.pmin[2]);
                        // periodic momentum neighbours of the column
                        const int cym = iy > 0 ? c - n2 : c + (n1 - 1) * n2, cyp = iy < n1 - 1 ? c + n2 : c - (n1 - 1) * n2;
                        const int czm = iz > 0 ? c - 1 : c + n2 - 1, czp = iz < n2 - 1 ? c + 1 : c - (n2 - 1);
#pragma unroll 2
                        for (int i = 0; i < n0; ++i) {
                            const int base = i * nyz, j = base + c;
                            const double iE = iEs[j];
                            const double vx = px_tab[i] * iE, vy = py * iE, vz = pz * iE;
                            const double Fx = fma(vy, QBz, fma(-vz, QBy, QEx));
                            const double Fy = fma(vz, QBx, fma(-vx, QBz, QEy));
                            const double Fz = fma(vx, QBy, fma(-vy, QBx, QEz));
                            const double c0d = fabs(Fx) * k0, c1d = fabs(Fy) * k1, c2d = fabs(Fz) * k2;
                            const int jxm = i > 0 ? j - nyz : j + (n0 - 1) * nyz, jxp = i < n0 - 1 ? j + nyz : j - (n0 - 1) * nyz;
                            const double self = fc[j];
                            const double u0 = fc[Fx > 0.0 ? jxm : jxp];
                            const double u1 = fc[base + (Fy > 0.0 ? cym : cyp)];
                            const double u2 = fc[base + (Fz > 0.0 ? czm : czp)];
                            const double num = fma(c2d, u2, fma(c1d, u1, fma(c0d, u0, self * (1.0 / 3.0))));
                            const double den = ((1.0 / 3.0 + c0d) + c1d) + c2d;
                            __stcs(oc + j, num * rcp_fast(den));          // den >= 1/3: no range checks; ~1 ulp
                        }
                    }
                }
            }
        }
        RBG_CHECK_STAGE(fs, f_species + (size_t)first * np, (size_t)cells * np);
        // no CTA barrier: a warp that is done moves on to the next stage; the last warp to finish with this one (its
        // shared-memory reads have completed: their values were consumed by the stores above) refills it
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            if (atomicAdd(&done[slot], 1) == MOM_THREADS / 32 - 1) {
                done[slot] = 0;
                arm(slot, u + n_stages * gridDim.x);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Vlasov step on a momentum grid symmetric about p = 0 (every workload of the paper), one spatial cell per stage.
// Same update as vlasov_upfd_kernel; differences:
//   * octant 1/E table (8 KB instead of 64 KB at 20^3): the ring has three stages;
//   * a column (ipy, ipz) is split into VS segments along ipx, one thread per (segment, column): 800 threads = 25 warps
//     at 20^3 where the column-per-thread kernel keeps 12.5 of its 16 warps busy (the kernel is latency-bound: 47 % issue
//     utilisation in round 1), at <= 80 registers;
//   * a thread always owns the same column and segment, so everything that depends on the momentum cell's (ipy, ipz) is
//     computed once per kernel; per spatial cell the force is built from pre-scaled fields,
//       c_x = dt |F_x| / dp_x = | e Ax + Ex' |,  Ax = k0 Q (p_y B_z - p_z B_y),  Ex' = k0 Q E_x,  e = 1 / E_p,
//       c_y = | e (Ay - p_x Bz') + Ey' |,  c_z = | e (p_x By' - Az) + Ez' |     (k_d = dt / dp_d folded into the constants),
//     5 FMAs per cell instead of 3 multiplies, 6 FMAs and 3 scalings.
// Every warp consumes every unit; the last warp to finish with a stage re-arms it (as in vlasov_upfd_kernel).
// ---------------------------------------------------------------------------------------------------------------
enum { VS_MAX_THREADS = 800, VS_STAGES = 3 };
struct __align__(16) VsPlane { double px; int erow; int pad; };   // per ipx: p_x and the byte offset of its row in the octant table

__global__ void __launch_bounds__(VS_MAX_THREADS, 1)
vlasov_sym_kernel(const double* __restrict__ f_species, double* __restrict__ out_species, SpeciesTables tb, VlasovParams vp,
                  int segs, int seg_len) {
    extern __shared__ __align__(128) unsigned char mom_smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(mom_smem);                             // VS_STAGES mbarriers
    int* done = reinterpret_cast<int*>(mom_smem + 64);                                  // [VS_STAGES] warps done with the stage
    VsPlane* xtab = reinterpret_cast<VsPlane*>(mom_smem + 128);                         // [n0]
    const int n0 = tb.n[0], n1 = tb.n[1], n2 = tb.n[2], nyz = n1 * n2;
    const int c0 = n0 >> 1, odd0 = n0 & 1, c1 = n1 >> 1, odd1 = n1 & 1, c2 = n2 >> 1, odd2 = n2 & 1;
    const int n0h = c0 + odd0, n1h = c1 + odd1, n2h = c2 + odd2, nyzh = n1h * n2h;
    double* iEc = reinterpret_cast<double*>(xtab + n0);                                 // [n0h][n1h][n2h] 1/E of one octant
    const size_t np = (size_t)tb.np;
    const size_t head = (128 + (size_t)n0 * 16 + (size_t)n0h * nyzh * 8 + 127) & ~(size_t)127;
    // a stage = [plane n0-1][the cell's n0 planes][plane 0]: the periodic p_x neighbours of the first and the
    // last plane are read like any other, without index wrapping in the loop
    const uint32_t plane_bytes = (uint32_t)nyz * 8u;
    const size_t stage_bytes = (np * 8 + 2 * (size_t)plane_bytes + 127) & ~(size_t)127;
    unsigned char* ring = mom_smem + head;
    const int lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int n_units = (vp.nx_cells - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto arm = [&](int slot, int k) {
        if (k < n_units) {
            const double* src = f_species + ((size_t)blockIdx.x + (size_t)k * gridDim.x) * np;
            unsigned char* dst = ring + (size_t)slot * stage_bytes;
            mbar_expect_tx(&bars[slot], (uint32_t)(np * 8) + 2u * plane_bytes);
            tma_bulk_g2s(dst + plane_bytes, src, (uint32_t)(np * 8), &bars[slot]);
            tma_bulk_g2s(dst, src + (np - (size_t)nyz), plane_bytes, &bars[slot]);
            tma_bulk_g2s(dst + plane_bytes + np * 8, src, plane_bytes, &bars[slot]);
        }
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < VS_STAGES; ++k) { mbar_init(&bars[k], 1); done[k] = 0; }
        fence_mbar_init();
        for (int k = 0; k < VS_STAGES; ++k) arm(k, k);
    }
    // rows 0 .. c0-1 of the octant table: the planes above the centre; row c0 (odd n only): the centre plane; likewise in
    // y and z (as in moments_sym_kernel)
    for (int i = threadIdx.x; i < n0; i += blockDim.x) {
        const int mi = i >= c0 + odd0 ? i - c0 - odd0 : (i < c0 ? c0 - 1 - i : c0);
        xtab[i].px = cell_centre(i, tb.delta[0], tb.pmin[0]);
        xtab[i].erow = mi * nyzh * 8;
        xtab[i].pad = 0;
    }
    for (int i = threadIdx.x; i < n0h * nyzh; i += blockDim.x) {
        const int j0 = i / nyzh, r = i - j0 * nyzh, j1 = r / n2h, j2 = r - j1 * n2h;
        const int i0 = j0 < c0 ? c0 + odd0 + j0 : c0, i1 = j1 < c1 ? c1 + odd1 + j1 : c1, i2 = j2 < c2 ? c2 + odd2 + j2 : c2;
        iEc[i] = __ldg(tb.iE + ((size_t)i0 * n1 + i1) * n2 + i2);
    }
    // this thread's (segment, column): fixed for the whole kernel
    const int seg = (int)threadIdx.x / nyz, c = (int)threadIdx.x - seg * nyz;
    const bool active = seg < segs;
    const int i_lo = min(seg * seg_len, n0), i_hi = active ? min(i_lo + seg_len, n0) : i_lo;
    const int iy = c / n2, iz = c - iy * n2;
    const double py = cell_centre(iy, tb.delta[1], tb.pmin[1]);
    const double pz = cell_centre(iz, tb.delta[2], tb.pmin[2]);
    // byte offsets of the periodic p_y, p_z neighbours relative to the cell itself (the same in every plane)
    const int dym = (iy > 0 ? -n2 : (n1 - 1) * n2) * 8, dyp = (iy < n1 - 1 ? n2 : -(n1 - 1) * n2) * 8;
    const int dzm = (iz > 0 ? -1 : n2 - 1) * 8, dzp = (iz < n2 - 1 ? 1 : -(n2 - 1)) * 8;
    const int m1 = iy >= c1 + odd1 ? iy - c1 - odd1 : (iy < c1 ? c1 - 1 - iy : c1);
    const int m2 = iz >= c2 + odd2 ? iz - c2 - odd2 : (iz < c2 ? c2 - 1 - iz : c2);
    const unsigned char* __restrict__ pe = reinterpret_cast<const unsigned char*>(iEc + m1 * n2h + m2);
    const double k0 = vp.dt / tb.delta[0], k1 = vp.dt / tb.delta[1], k2 = vp.dt / tb.delta[2];
    const double Q = tb.charge;
    const double third = 1.0 / 3.0;
    const size_t j_lo = (size_t)i_lo * nyz + c;
    __syncthreads();
    uint32_t phases = 0;
    for (int k = 0; k < n_units; ++k) {
        const int slot = k % VS_STAGES;
        const size_t cell = (size_t)blockIdx.x + (size_t)k * gridDim.x;
        const unsigned char* __restrict__ fcb = ring + (size_t)slot * stage_bytes + plane_bytes;    // plane 0 of the cell
        // F = Q (E + v x B); Q and dt / dp_d folded into the fields of this spatial cell
        const double* __restrict__ Ev = vp.E + cell * 3;
        const double* __restrict__ Bv = vp.B + cell * 3;
        const double QBx = Q * __ldg(Bv), QBy = Q * __ldg(Bv + 1), QBz = Q * __ldg(Bv + 2);
        const double Ex = k0 * (Q * __ldg(Ev)), Ey = k1 * (Q * __ldg(Ev + 1)), Ez = k2 * (Q * __ldg(Ev + 2));
        const double Ax = k0 * fma(py, QBz, -(pz * QBy));               // k0 Q E_p (v x B)_x
        const double Ay = k1 * (pz * QBx), Bz1 = k1 * QBz;              // k1 Q E_p (v x B)_y = Ay - p_x Bz1
        const double Az = k2 * (py * QBx), By2 = k2 * QBy;              // k2 Q E_p (v x B)_z = p_x By2 - Az
        mbar_wait(&bars[slot], (phases >> slot) & 1u);
        phases ^= 1u << slot;
        RBG_CHECK_STAGE(reinterpret_cast<const double*>(fcb), f_species + cell * np, np);
        RBG_CHECK(cell < (size_t)vp.nx_cells && (size_t)(slot + 1) * stage_bytes + head <= dynamic_smem_size(), CHK_BE_INDEX);
        // walk up the segment with the p_x neighbours in registers: one load brings the next plane's value
        const unsigned char* __restrict__ a = fcb + j_lo * 8;
        double* __restrict__ op = out_species + cell * np + j_lo;
        double prev = *reinterpret_cast<const double*>(a - plane_bytes);
        double cur = active ? *reinterpret_cast<const double*>(a) : 0.0;
#pragma unroll 2
        for (int i = i_lo; i < i_hi; ++i) {
            const double next = *reinterpret_cast<const double*>(a + plane_bytes);
            const VsPlane xp = xtab[i];
            const double e = *reinterpret_cast<const double*>(pe + xp.erow);
            const double Fx = fma(e, Ax, Ex);
            const double Fy = fma(e, fma(-xp.px, Bz1, Ay), Ey);
            const double Fz = fma(e, fma(xp.px, By2, -Az), Ez);
            const double u0 = Fx > 0.0 ? prev : next;
            const double u1 = *reinterpret_cast<const double*>(a + (Fy > 0.0 ? dym : dyp));
            const double u2 = *reinterpret_cast<const double*>(a + (Fz > 0.0 ? dzm : dzp));
            const double cxd = fabs(Fx), cyd = fabs(Fy), czd = fabs(Fz);
            const double num = fma(czd, u2, fma(cyd, u1, fma(cxd, u0, cur * third)));
            const double den = ((third + cxd) + cyd) + czd;
            __stcs(op, num * rcp_fast(den));                             // den >= 1/3: no range checks; ~1 ulp
            prev = cur; cur = next;
            a += plane_bytes; op += nyz;
        }
        RBG_CHECK_STAGE(reinterpret_cast<const double*>(fcb), f_species + cell * np, np);
        // the last warp to finish with this stage (its shared-memory reads have completed: their values were consumed by
        // the stores above) refills it
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            if (atomicAdd(&done[slot], 1) == nwarps - 1) {
                done[slot] = 0;
                arm(slot, k + VS_STAGES);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Direct (unstaged) variants for momentum grids whose block of one spatial cell does not fit in shared memory twice
// (e.g. the paper's 35^3 test grid, 343 KB): same arithmetic, f read straight from global memory / L2.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
moments_direct_kernel(const double* __restrict__ f_species, SpeciesTables tb, int nx_cells, double* __restrict__ M_species) {
    __shared__ double red[4][N_MOMENTS];
    const int ix = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const double* __restrict__ f = f_species + (size_t)ix * tb.np;
    const double* __restrict__ iE = tb.iE;
    const int nyz = tb.n[1] * tb.n[2];
    const double msq = tb.mass * tb.mass;
    double acc[N_MOMENTS];
#pragma unroll
    for (int m = 0; m < N_MOMENTS; ++m) acc[m] = 0.0;
    for (int c = warp * 32 + lane; c < nyz; c += nwarps * 32) {
        const int iy = c / tb.n[2], iz = c - iy * tb.n[2];
        const double py = cell_centre(iy, tb.delta[1], tb.pmin[1]);
        const double pz = cell_centre(iz, tb.delta[2], tb.pmin[2]);
        double X0 = 0.0, X1 = 0.0, G0 = 0.0, G1 = 0.0, G2 = 0.0;
#pragma unroll 4
        for (int i = 0; i < tb.n[0]; ++i) {
            const double px = cell_centre(i, tb.delta[0], tb.pmin[0]);
            const size_t j = (size_t)i * nyz + c;
            const double a = __ldcs(f + j);
            const double g = a * __ldg(iE + j);
            const double pg = px * g;
            X0 += a;
            X1 = fma(px, a, X1);
            G0 += g;
            G1 += pg;
            G2 = fma(px, pg, G2);
        }
        const double r = fma(py, py, fma(pz, pz, msq));
        const double yG0 = py * G0, zG0 = pz * G0;
        acc[0] += X0;
        acc[1] += G1; acc[2] += yG0; acc[3] += zG0;
        acc[4] += fma(r, G0, G2);
        acc[5] += X1; acc[6] = fma(py, X0, acc[6]); acc[7] = fma(pz, X0, acc[7]);
        acc[8] += G2; acc[9] = fma(py, G1, acc[9]); acc[10] = fma(pz, G1, acc[10]);
        acc[11] = fma(py, yG0, acc[11]); acc[12] = fma(py, zG0, acc[12]); acc[13] = fma(pz, zG0, acc[13]);
    }
#pragma unroll
    for (int m = 0; m < N_MOMENTS; ++m) {
        double v = acc[m];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][m] = v;
    }
    __syncthreads();
    if (threadIdx.x < N_MOMENTS) {
        double v = 0.0;
        for (int w = 0; w < nwarps; ++w) v += red[w][threadIdx.x];
        M_species[(size_t)ix * N_MOMENTS + threadIdx.x] = v * (tb.delta[0] * tb.delta[1] * tb.delta[2]);
    }
}

// thread = one momentum cell (velocity in registers), walking over `slab` consecutive spatial cells
__global__ void __launch_bounds__(256)
vlasov_direct_kernel(const double* __restrict__ f_species, double* __restrict__ out_species, SpeciesTables tb, VlasovParams vp, int slab) {
    const int nchunks = (tb.np + blockDim.x - 1) / blockDim.x;
    const int chunk = blockIdx.x % nchunks, sl = blockIdx.x / nchunks;
    const int ip = chunk * blockDim.x + threadIdx.x;
    if (ip >= tb.np) return;
    const int ix_begin = sl * slab, ix_end = min(ix_begin + slab, vp.nx_cells);
    const int nyz = tb.n[1] * tb.n[2];
    const int i0 = ip / nyz, i1 = (ip - i0 * nyz) / tb.n[2], i2 = ip - i0 * nyz - i1 * tb.n[2];
    // periodic momentum neighbours: m at p_d - dp_d, p at p_d + dp_d
    const int x_m = ip + (i0 > 0 ? -nyz : (tb.n[0] - 1) * nyz), x_p = ip + (i0 < tb.n[0] - 1 ? nyz : -(tb.n[0] - 1) * nyz);
    const int y_m = ip + (i1 > 0 ? -tb.n[2] : (tb.n[1] - 1) * tb.n[2]), y_p = ip + (i1 < tb.n[1] - 1 ? tb.n[2] : -(tb.n[1] - 1) * tb.n[2]);
    const int z_m = ip + (i2 > 0 ? -1 : tb.n[2] - 1), z_p = ip + (i2 < tb.n[2] - 1 ? 1 : -(tb.n[2] - 1));
    // the same v = p * (1/E) as the staged kernel
    const double iE = __ldg(tb.iE + ip);
    const double vx = cell_centre(i0, tb.delta[0], tb.pmin[0]) * iE;
    const double vy = cell_centre(i1, tb.delta[1], tb.pmin[1]) * iE;
    const double vz = cell_centre(i2, tb.delta[2], tb.pmin[2]) * iE;
    const double k0 = vp.dt / tb.delta[0], k1 = vp.dt / tb.delta[1], k2 = vp.dt / tb.delta[2];
    const double Q = tb.charge;
    const size_t np = (size_t)tb.np;
    for (int ix = ix_begin; ix < ix_end; ++ix) {
        const double* __restrict__ row = f_species + (size_t)ix * np;
        const double* __restrict__ Ev = vp.E + (size_t)ix * 3;
        const double* __restrict__ Bv = vp.B + (size_t)ix * 3;
        const double QEx = Q * __ldg(Ev), QEy = Q * __ldg(Ev + 1), QEz = Q * __ldg(Ev + 2);
        const double QBx = Q * __ldg(Bv), QBy = Q * __ldg(Bv + 1), QBz = Q * __ldg(Bv + 2);
        const double Fx = fma(vy, QBz, fma(-vz, QBy, QEx));
        const double Fy = fma(vz, QBx, fma(-vx, QBz, QEy));
        const double Fz = fma(vx, QBy, fma(-vy, QBx, QEz));
        const double c0 = fabs(Fx) * k0, c1 = fabs(Fy) * k1, c2 = fabs(Fz) * k2;
        const double self = __ldg(row + ip);
        const double u0 = __ldg(row + (Fx > 0.0 ? x_m : x_p));
        const double u1 = __ldg(row + (Fy > 0.0 ? y_m : y_p));
        const double u2 = __ldg(row + (Fz > 0.0 ? z_m : z_p));
        const double num = fma(c2, u2, fma(c1, u1, fma(c0, u0, self * (1.0 / 3.0))));
        const double den = ((1.0 / 3.0 + c0) + c1) + c2;
        __stcs(out_species + (size_t)ix * np + ip, num * rcp_fast(den));
    }
}

}  // namespace rbg
