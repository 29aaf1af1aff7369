// rbg_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, scalar CPU oracle for the Monte Carlo evaluation of the relativistic 2->2
// Boltzmann collision term C_a[f](x,p1) (Eq. 16; quantum factor Eq. 18
// PAPER.md:192-197; species sum and symmetry factor Eq. 19).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code, header, table or constant generator with
// the CUDA path under paper_2308_04869_b200/csrc and neither includes the other.
//
// What it computes.  Eq. 16 for "a(k1)+b(k2)->c(k3)+d(p)" with the grid particle d(p)==p1, its
// partner c(k3)==p2 and the other pair (k1,k2)==(p3,p4).  Integrating d3p3 d3p4 delta4/(E3 E4) by
// two-body phase space (= |p*|/sqrt(s) dOmega*) leaves the reduced form (R) of DESIGN.md section 2:
//
//   C_role(x,p1) = sym * Int_box(s2) d3p2 Int_4pi dOmega*  |M|^2 |p*_34| / (64 pi^2 E1 E2 sqrt(s))
//                        * [ f3 f4 F1 F2  -  f1 f2 F3 F4 ],          F = 1 + theta (2 pi hbar)^3 f / g
//
// which is estimated with N samples: p2 uniform in the species-2 momentum box (volume V2), the
// CM direction n uniform on the sphere, so C_role ~= sym V2 4pi / N * Sum integrand
//          = sym V2 / (16 pi E1 N) * Sum  w (gain - loss),   w = |M|^2 |p*| / (E2 sqrt(s)).
//
// The paper leaves sampler, RNG and arithmetic order to an external package, so
// the step-by-step chain below (O0..O14) is the reading fixed in DESIGN.md section 4; every
// floating-point operation up to a cell-index decision is written as ONE IEEE operation
// (fma() = one rounding; every other operator one rounding; no contraction: build with
// -ffp-contract=off) so that an independent implementation can reproduce the decisions exactly.
//
// Pins (tests/test_oracle_*.py): Philox known answers, per-sample kinematic invariants, the
// massless closed form, a scipy quadrature of the loss rate, exact detailed balance for
// MJ/FD/BE inputs, the paper's own 5-D form Eq. 37 (oracle/eq37.py), number/energy conservation,
// deterministic brute-force quadrature of (R) (oracle/quadrature.py), H-theorem sign,
// thread-count independence; Table III kinds against textbook values, crossing symmetry and regulator limits;
// inelastic roles against per-sample kinematics, detailed balance, the quadrature and cross-species bookkeeping
// (tests/test_oracle_qcd.py).  PARITY UNPINNED (by the reference): orc_collision_symmetric -- the paper names the
// "symmetric sampling method [57]" but defines it outside PAPER.md; it is pinned by invariants only
// (tests/test_oracle_symmetric.py).  Every other function here is pinned.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <string>
#include <type_traits>
#include <map>
#include <utility>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------------
// O1. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  Counter-based: out = P(key, counter).
// ---------------------------------------------------------------------------------------------
struct U4 { uint32_t v[4]; };

inline U4 philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // round multipliers
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl key increments
    for (int round = 0; round < 10; ++round) {
        const uint64_t prod0 = (uint64_t)M0 * c0;
        const uint64_t prod1 = (uint64_t)M1 * c2;
        const uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
        const uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    return U4{{c0, c1, c2, c3}};
}

// ---------------------------------------------------------------------------------------------
// Problem description (mirrors what the caller passes; plain structs, C layout)
// ---------------------------------------------------------------------------------------------
struct Species { double mass, charge; int stat; double g; };
struct Grid    { int n[3]; double pmin[3], pmax[3]; };
struct Process { int a, b, c, d; int kind; double par[4]; double sym; int sampler; };

enum Kind { M2_CONST = 0, M2_COULOMB_SCREENED = 1, M2_TCHAN_S2 = 2,
            // |M|^2 = 64 pi^2 s par0: a constant differential cross section dsigma/dOmega = par0, isotropic in
            // the CM frame (the paper's collision test quotes its processes this way, Eq. 48 PAPER.md:493-500;
            // relation cross section <-> matrix element: Eq. 20-22, reading R17)
            M2_ISO_DSIGMA = 3,
            // Table III: |M|^2 of the 2->2 parton processes of QCD, summed over the helicities and
            // colours of all four particles, with the regulator m_g^2 = par1^2 subtracted from t and u in the
            // denominators; g = par0; SU_c(3): d_F = C_A = 3, C_F = 4/3, d_A = 8.  t = (p1-p3)^2, u = (p1-p4)^2
            // (role labels; the role permutations of orc_create keep t and u those of the process as written).
            // Rows :677, :679, :683-684 and :687 of the table are garbled in PAPER.md: they are restated from the
            // legible rows by crossing symmetry (reading R20) and all rows are pinned to the textbook
            // 90-degree values (tests/golden/qcd_90deg.txt).
            M2_QCD_Q1Q2 = 4,           // q1 q2 -> q1 q2 (also qbar1 q2, q1 qbar2, qbar1 qbar2)
            M2_QCD_Q1Q1 = 5,           // q1 q1 -> q1 q1 (also qbar1 qbar1)
            M2_QCD_Q1QB1 = 6,          // q1 qbar1 -> q1 qbar1
            M2_QCD_Q1QB1_Q2QB2 = 7,    // q1 qbar1 -> q2 qbar2
            M2_QCD_QQB_GG = 8,         // q1 qbar1 -> g g
            M2_QCD_QG = 9,             // q1 g -> q1 g (also qbar1 g)
            M2_QCD_GG = 10,            // g g -> g g
            M2_KIND_LAST = 10 };

// A role = one process seen from one grid species: particle 1 is the grid
// particle, 2 its sampled partner, (3,4) the other pair.
// sampler: how the CM scattering direction is drawn.  0 = uniform on the sphere (O6); 1 = polar angle
// about the CM direction of particle 1 drawn from the t-channel shape 1/(t - mD^2)^2 by its inverse CDF
// (steps S1..S7 below), azimuth uniform.  Both estimate the same integral (R).
enum Sampler { SAMPLER_UNIFORM = 0, SAMPLER_TCHANNEL = 1 };
struct Role { int s[4]; int kind; double par[4]; double sym; int process; int sampler; double gab; double sym_override; };

typedef double (*FCallback)(int species, const double* p, void* user);

// Built-in analytic input family for analytic-f mode (an INPUT, not part of the method):
//   f_s(p) = scale / ( exp((sqrt(|p-u|^2 + m^2) - mu)/T) - theta ),  8 doubles per species in
// `user`: scale, T, mu, m, theta, ux, uy, uz.  theta=0: Maxwell-Juttner (Eq. 11),
// -1/+1: Fermi-Dirac / Bose-Einstein occupation times scale.
extern "C" double orc_builtin_thermal(int species, const double* p, void* user) {
    const double* q = (const double*)user + 8 * species;
    const double dx = p[0] - q[5], dy = p[1] - q[6], dz = p[2] - q[7];
    const double E = std::sqrt(dx * dx + dy * dy + dz * dz + q[3] * q[3]);
    return q[0] / (std::exp((E - q[2]) / q[1]) - q[4]);
}

struct Handle {
    int nx = 0;
    std::vector<Species> sp;
    std::vector<Grid> grid;
    std::vector<Role> roles;
    std::vector<size_t> sp_off;     // offset of species s in the f / C arrays
    std::vector<size_t> np;         // momentum cells of species s
    std::vector<size_t> role_off;   // offset of role r in the per-role detail arrays
    double hbar = 1.0;
    int use_float = 0;
    std::string err;
};

// Per-sample record for tests (oracle-only).
struct Trace {
    double p1[3], p2[3], p3[3], p4[3];
    double E1, E2, E3, s, t, pf, w, f1, f2, f3, f4, gain, loss, u;
    int j2, j3, j4;            // linear momentum cell, -1 = outside the box
    int status;                // 0 ok, 1 skipped at O4 (h<=0), 2 below threshold
    int draws;                 // Philox calls consumed (always 1)
};


template <typename R> inline R rfma(R a, R b, R c);
template <> inline double rfma<double>(double a, double b, double c) { return std::fma(a, b, c); }
template <> inline float  rfma<float>(float a, float b, float c) { return std::fmaf(a, b, c); }

// O2: top 24 bits of a word -> uniform real in [0,1), exact in both types.
template <typename R> inline R u01(uint32_t x) { return (R)(x >> 8) * (R)0x1p-24; }
// O6: a word -> uniform real in [-1,1): double keeps all 32 bits, float the top 24; both exact.
template <typename R> inline R usym(uint32_t x);
template <> inline double usym<double>(uint32_t x) { return (double)x * 0x1p-31 - 1.0; }
template <> inline float  usym<float>(uint32_t x) { return (float)(x >> 8) * 0x1p-23f - 1.0f; }

// O6: cos and sin of an angle a in (0, pi/4) as fixed polynomials in z = a*a, Horner with fma.
// The coefficients are part of the chain (table "direction polynomials"):
// near-minimax fits of (sin(a)/a - 1)/z and (cos(a) - 1)/z on [0, (pi/4)^2]; absolute error
// <= 3e-16 (double, 6 terms each) and <= 1.5e-7 (float, 3 and 4 terms).
template <typename R> struct OctantPoly;
template <> struct OctantPoly<double> {
    static void eval(double a, double& ca, double& sa) {
        const double S1 = -0x1.5555555555555p-3, S2 = 0x1.1111111110bb2p-7, S3 = -0x1.a01a019e83aaep-13,
                     S4 = 0x1.71de37968a100p-19, S5 = -0x1.ae600b02b6262p-26, S6 = 0x1.5e0b19f8b1451p-33;
        const double C1 = -0x1.ffffffffffffap-2, C2 = 0x1.5555555554137p-5, C3 = -0x1.6c16c1691d8abp-10,
                     C4 = 0x1.a019fc7b4b9f6p-16, C5 = -0x1.27e0f5789db4bp-22, C6 = 0x1.1c064801aa169p-29;
        const double z = a * a;
        double ps = std::fma(S6, z, S5); ps = std::fma(ps, z, S4); ps = std::fma(ps, z, S3);
        ps = std::fma(ps, z, S2); ps = std::fma(ps, z, S1);
        sa = std::fma(a * z, ps, a);
        double pc = std::fma(C6, z, C5); pc = std::fma(pc, z, C4); pc = std::fma(pc, z, C3);
        pc = std::fma(pc, z, C2); pc = std::fma(pc, z, C1);
        ca = std::fma(z, pc, 1.0);
    }
};
template <> struct OctantPoly<float> {
    static void eval(float a, float& ca, float& sa) {
        const float S1 = -0x1.555552p-3f, S2 = 0x1.110c28p-7f, S3 = -0x1.9ac9bp-13f;
        const float C1 = -0x1p-1f, C2 = 0x1.55554cp-5f, C3 = -0x1.6c0e08p-10f, C4 = 0x1.9a6f2cp-16f;
        const float z = a * a;
        float ps = std::fmaf(S3, z, S2); ps = std::fmaf(ps, z, S1);
        sa = std::fmaf(a * z, ps, a);
        float pc = std::fmaf(C4, z, C3); pc = std::fmaf(pc, z, C2); pc = std::fmaf(pc, z, C1);
        ca = std::fmaf(z, pc, 1.0f);
    }
};

// O6: unit vector, uniform on the sphere, from one word for cos(theta) and 24 bits for phi.
//   nz = usym(x3 | odd), odd = lowest bit that usym keeps (so |nz| < 1 and the lattice is symmetric);
//   sin(theta) = sqrt(1 - nz^2);
//   azimuth from the 24-bit integer k: quadrant q = k >> 22, second-half flag b = bit 21, in-octant index
//   r = k & (2^21 - 1), folded r' = b ? 2^21 - 1 - r : r; (cos, sin) of the angle a in (0, pi/4) inside the octant (below);
//   (cos, sin) of the angle inside the quadrant = b ? (sin a, cos a) : (cos a, sin a), then the exact rotation by q * pi/2.
// float chain:  a = (r' + 1/2)(pi/4)/2^21, cos a and sin a from the octant polynomials.
// double chain (chain v3): the lattice keeps the top 19 bits of r', r19 = r' >> 2 = 2^10 hi + lo, and the angle is split
//   a = alpha + beta,  alpha = (2^10 hi) A1,  beta = (lo + 1/2) A1,  A1 = (pi/4) / 2^19  (beta = fma(lo, A1, A1/2)),
//   cos a = cos(alpha) cos(beta) - sin(alpha) sin(beta),  sin a = sin(alpha) cos(beta) + cos(alpha) sin(beta),
//   each written as one fma of a product, with cos / sin of alpha and of beta from the octant polynomials (both angles
//   lie in [0, pi/4)).  alpha takes 512 values and beta 1024, so an implementation may tabulate the four factors.
template <typename R> inline void octant_angle(uint32_t rf21, R& ca, R& sa);
template <> inline void octant_angle<float>(uint32_t rf21, float& ca, float& sa) {
    const float A1 = (float)0x1.921fb54442d18p-22;       // (pi/4) / 2^21
    const float A0 = (float)0x1.921fb54442d18p-23;       // half a step
    OctantPoly<float>::eval(rfma<float>((float)rf21, A1, A0), ca, sa);
}
template <> inline void octant_angle<double>(uint32_t rf21, double& ca, double& sa) {
    const double A1 = 0x1.921fb54442d18p-20;             // (pi/4) / 2^19
    const double A0 = 0x1.921fb54442d18p-21;             // half a step
    const uint32_t r19 = rf21 >> 2, hi = r19 >> 10, lo = r19 & 1023u;
    double cA, sA, cB, sB;
    OctantPoly<double>::eval((double)(hi << 10) * A1, cA, sA);
    OctantPoly<double>::eval(std::fma((double)lo, A1, A0), cB, sB);
    ca = std::fma(cA, cB, -(sA * sB));
    sa = std::fma(sA, cB, cA * sB);
}
template <typename R> inline void azimuth(uint32_t k24, R& cphi, R& sphi) {
    const uint32_t q = k24 >> 22, b = (k24 >> 21) & 1u, r = k24 & 0x1FFFFFu;
    const uint32_t rf = b ? 0x1FFFFFu - r : r;
    R ca, sa;
    octant_angle<R>(rf, ca, sa);
    const R c1 = b ? sa : ca, s1 = b ? ca : sa;  // angle in (0, pi/2)
    switch (q) {
        case 0:  cphi = c1;  sphi = s1;  break;
        case 1:  cphi = -s1; sphi = c1;  break;
        case 2:  cphi = -c1; sphi = -s1; break;
        default: cphi = s1;  sphi = -c1; break;
    }
}
template <typename R> inline void direction(uint32_t x3, uint32_t k24, R nh[3]) {
    const R nz = usym<R>(x3 | (sizeof(R) == 8 ? 1u : 0x100u));   // odd lattice: symmetric, never +-1
    const R st = std::sqrt(rfma<R>(-nz, nz, (R)1));
    R cphi, sphi;
    azimuth<R>(k24, cphi, sphi);
    nh[0] = st * cphi; nh[1] = st * sphi; nh[2] = nz;
}

// O6 BY EYE -- not part of the chain, never called by the estimator.  direction() above reaches its lattice point through
// minimax polynomials, an octant fold and (double chain) an angle split chosen so that an implementation can tabulate it;
// none of that can be checked against the paper by reading it.  This is the same lattice point straight from the
// definition of a unit vector, n = (sin(theta) cos(phi), sin(theta) sin(phi), cos(theta)), with the C library's cosl / sinl
// in extended precision (x86-64 long double: 64-bit significand, so the result is the exact value rounded once, for the
// purposes of a 4e-16 comparison):
//   cos(theta) = (x3 | 1) 2^-31 - 1                    (double chain; float chain: ((x3 >> 8) | 1) 2^-23 - 1)
//   phi        = ((k24 >> 2) + 1/2) 2 pi / 2^22        (double chain; float chain: (k24 + 1/2) 2 pi / 2^24)
// tests/test_oracle_kinematics.py compares the two on every octant boundary and on random words.  The chain cannot use
// this form itself: libm results differ by an ulp between machines and the kernels must reproduce every cell-index
// decision bit for bit.
template <typename R> inline void direction_by_eye(uint32_t x3, uint32_t k24, double nh[3]) {
    const long double PI_L = 3.14159265358979323846264338327950288L;
    const bool dbl = sizeof(R) == 8;
    const long double ct = dbl ? (long double)(x3 | 1u) / 2147483648.0L - 1.0L : (long double)((x3 >> 8) | 1u) / 8388608.0L - 1.0L;
    const long double phi = dbl ? ((long double)(k24 >> 2) + 0.5L) * (2.0L * PI_L / 4194304.0L)
                                : ((long double)k24 + 0.5L) * (2.0L * PI_L / 16777216.0L);
    const long double st = sqrtl(1.0L - ct * ct);
    nh[0] = (double)(st * cosl(phi));
    nh[1] = (double)(st * sinl(phi));
    nh[2] = (double)ct;
}

// S2 (t-channel sampler): a word -> uniform real in (0,1) on the half-integer lattice, exact in both types:
// double (x + 1/2) 2^-32, float ((x >> 8) + 1/2) 2^-24.  uhalf(~x) = 1 - uhalf(x) exactly.
template <typename R> inline R uhalf(uint32_t x);
template <> inline double uhalf<double>(uint32_t x) { return std::fma((double)x, 0x1p-32, 0x1p-33); }
template <> inline float  uhalf<float>(uint32_t x) { return std::fmaf((float)(x >> 8), 0x1p-24f, 0x1p-25f); }

template <typename R> struct RoleConst {
    R m[4], msq[4];
    R m1m2, msum2, Mth, Mdf, dm34;
    R pmin[4][3], L[4][3], invD[4][3], off[4][3];   // per particle slot (its species' grid)
    int n[4][3];
    R theta_kappa[4];
    R par0, mD2, twomD2, g4, sig64;
    R msqsum;                      // m1^2 + m2^2 + m3^2 + m4^2 (u = msqsum - s - t)
    R qA, qB, qC, qD, qG;          // Table III group factors times g^4 (see Evaluator)
    R cg, cl;                      // degrees-of-freedom factors of the gain and the loss direction (see Evaluator)
};

template <typename R> inline R dot3(const R* a, const R* b) {
    return rfma<R>(a[2], b[2], rfma<R>(a[1], b[1], a[0] * b[0]));
}

struct Accum { double G = 0, Ls = 0, Lin = 0, Q = 0, D = 0; };

// NEXT-3, "symmetric" (conservative) sampling -- PAPER.md:257 names "the symmetric sampling method [57]" for the
// collision term but does not define it and Ref. [57] is not part of PAPER.md: PARITY UNPINNED BY THE REFERENCE
// (reading R25).  The reading implemented: every Monte Carlo sample is one sampled reaction 1+2 <-> 3+4
// with net rate q = pref0 * w (gain - loss); instead of crediting it to the grid particle alone it is credited to all
// four particles, +q to the cells of 1 and 2 and -q to the cells of 3 and 4, so that what one cell gains another
// loses, sample by sample.  Each of the four deposits is by itself an unbiased estimator of the collision term of
// its slot's species (two-body phase space is symmetric under (1,2) <-> (3,4)), so C of a species is their average.
// fac[k] = sigma_k * sym_k * (dp^3 of species 1 / dp^3 of slot k's species) / m, with sigma = (+,+,-,-), sym_k the
// symmetry factor seen from slot k (1/2 iff the opposite pair is one species) and m the number of (role, slot) pairs
// of the process that carry the slot's species.
struct SymSink { double* C; double* mag; double fac[4]; };   // D: float chain's sum of (float)(w gain - w loss)

template <typename R>
struct Evaluator {
    const Handle& H; const Role& role; int irole;
    RoleConst<R> k;
    FCallback fcb; void* user; int box_cut;   // analytic-f mode when fcb != nullptr

    Evaluator(const Handle& h, int ir, FCallback cb, void* u, int cut)
        : H(h), role(h.roles[ir]), irole(ir), fcb(cb), user(u), box_cut(cut) {
        // Role constants: computed in double by the formulas below, then rounded to R.
        double m[4];
        for (int i = 0; i < 4; ++i) m[i] = H.sp[role.s[i]].mass;
        for (int i = 0; i < 4; ++i) { k.m[i] = (R)m[i]; k.msq[i] = (R)(m[i] * m[i]); }
        const double msum = m[0] + m[1], m34 = m[2] + m[3], md = m[2] - m[3];
        k.m1m2  = (R)(m[0] * m[1]);
        k.msum2 = (R)(msum * msum);
        k.Mth   = (R)(msum * msum - m34 * m34);
        k.Mdf   = (R)(md * md);
        k.dm34  = (R)(m[2] * m[2] - m[3] * m[3]);
        const double twopihbar = 2.0 * M_PI * H.hbar;
        for (int i = 0; i < 4; ++i) {
            const Grid& g = H.grid[role.s[i]];
            for (int d = 0; d < 3; ++d) {
                const double L = g.pmax[d] - g.pmin[d];
                const double invD = (double)g.n[d] / L;
                k.n[i][d] = g.n[d];
                k.pmin[i][d] = (R)g.pmin[d];
                k.L[i][d] = (R)L;
                k.invD[i][d] = (R)invD;
                k.off[i][d] = (R)(-g.pmin[d] * invD);
            }
            const Species& S = H.sp[role.s[i]];
            k.theta_kappa[i] = (R)((double)S.stat * (twopihbar * twopihbar * twopihbar) / S.g);
        }
        k.par0 = (R)role.par[0];
        k.mD2  = (R)(role.par[1] * role.par[1]);
        k.twomD2 = (R)(2.0 * (role.par[1] * role.par[1]));
        const double g2 = role.par[0] * role.par[0];
        k.g4   = (R)(g2 * g2);
        k.sig64 = (R)(64.0 * M_PI * M_PI * role.par[0]);     // M2_ISO_DSIGMA: |M|^2 = sig64 * s
        k.msqsum = (R)((m[0] * m[0] + m[1] * m[1]) + (m[2] * m[2] + m[3] * m[3]));
        // Table III prefactors (d_F = C_A = 3, C_F = 4/3, d_A = 8), times g^4 = par0^4
        const double dF = 3.0, CA = 3.0, CF = 4.0 / 3.0, dA = 8.0, g4d = g2 * g2;
        k.qA = (R)(8.0 * g4d * dF * dF * CF * CF / dA);          // 8 g^4 dF^2 CF^2 / dA
        k.qB = (R)(16.0 * g4d * dF * CF * (CF - CA / 2.0));      // 16 g^4 dF CF (CF - CA/2)
        k.qC = (R)(8.0 * g4d * dF * CF * CF);                    // 8 g^4 dF CF^2
        k.qD = (R)(8.0 * g4d * dF * CF * CA);                    // 8 g^4 dF CF CA
        k.qG = (R)(16.0 * g4d * dA * CA * CA);                   // 16 g^4 dA CA^2
        // Degrees of freedom ("an average over the DOF in the initial state and a sum over the DOF
        // in the final state are implied in M_{ab<->cd}, and a sum over the DOF of the distribution function is
        // also implied"; reading R21).  With |M|^2_sum the matrix element summed over the DOF of all
        // four particles, the loss direction 1+2 -> 3+4 carries |M|^2_sum / (g1 g2) and the gain direction
        // 3+4 -> 1+2 carries |M|^2_sum / (g3 g4).  Table III kinds ARE |M|^2_sum; kinds 0..3
        // give |M|^2 of the process as written, a+b -> c+d, averaged over g_a g_b, i.e. |M|^2_sum = |M|^2 g_a g_b.
        // For an elastic role of kinds 0..3 both factors are exactly 1.
        {
            const Process_dof d = dof_of(H, role);
            k.cl = (R)(d.sum_norm / (d.g[0] * d.g[1]));
            k.cg = (R)(d.sum_norm / (d.g[2] * d.g[3]));
        }
    }

    struct Process_dof { double g[4]; double sum_norm; };
    static Process_dof dof_of(const Handle& h, const Role& r) {
        Process_dof d;
        for (int i = 0; i < 4; ++i) d.g[i] = h.sp[r.s[i]].g;
        d.sum_norm = r.kind >= M2_QCD_Q1Q2 ? 1.0 : r.gab;      // gab = g_a g_b of the process as written
        return d;
    }

    // O9 for the Table III kinds: |M|^2(s,t,u) with T = t - m_g^2, U = u - m_g^2.
    inline R m2_qcd(R s, R t, R u) const {
        const R T = t - k.mD2, U = u - k.mD2;
        const R s2 = s * s, t2 = t * t, u2 = u * u;
        switch (role.kind) {
            case M2_QCD_Q1Q2:        return k.qA * ((s2 + u2) / (T * T));
            case M2_QCD_Q1Q1:        return k.qA * ((s2 + u2) / (T * T) + (s2 + t2) / (U * U)) + k.qB * (s2 / (T * U));
            case M2_QCD_Q1QB1:       return k.qA * ((s2 + u2) / (T * T) + (u2 + t2) / s2) + k.qB * (u2 / (T * s));
            case M2_QCD_Q1QB1_Q2QB2: return k.qA * ((t2 + u2) / s2);
            case M2_QCD_QQB_GG:      return k.qC * (u / T + t / U) - k.qD * ((t2 + u2) / s2);
            case M2_QCD_QG:          return k.qD * ((s2 + u2) / (T * T)) - k.qC * (u / s + s / U);
            default:                 return k.qG * ((((R)3 - (s * u) / (T * T)) - (s * t) / (U * U)) - (t * u) / s2);
        }
    }

    // O10.  Nearest-cell gather: tau_d = fma(p_d, invDelta_d, -pmin_d*invDelta_d); inside iff
    // 0 <= floor(tau_d) < n_d for all d; zero outside the box (north_star).  Returns cell or -1.
    inline int cell_of(int slot, const R* p) const {
        int j[3];
        for (int d = 0; d < 3; ++d) {
            const R tau = rfma<R>(p[d], k.invD[slot][d], k.off[slot][d]);
            const R fl = std::floor(tau);
            if (!(fl >= (R)0) || !(fl < (R)k.n[slot][d])) return -1;
            j[d] = (int)fl;
        }
        return (j[0] * k.n[slot][1] + j[1]) * k.n[slot][2] + j[2];
    }

    // One p1: N samples.  The f value of species s, spatial cell ix, momentum cell j is
    // f_all[sp_off[s] + ix*np[s] + j] (layout of DESIGN.md section 5).
    void eval_p1(const double* f_all, int ix, int ip1, int N, uint64_t seed, Accum& acc, Trace* trace,
                 int trace_n, const SymSink* sink = nullptr) const {
        const uint32_t key0 = (uint32_t)seed, key1 = (uint32_t)(seed >> 32);
        // species table base pointers at this spatial cell (index = sp_off[s] + ix*np[s])
        auto fval = [&](int slot, int cell, const R* p) -> R {
            if (fcb) {
                if (box_cut && cell < 0) return (R)0;
                const double pd[3] = {(double)p[0], (double)p[1], (double)p[2]};
                return (R)fcb(role.s[slot], pd, user);
            }
            if (cell < 0) return (R)0;
            const int s = role.s[slot];
            return (R)f_all[H.sp_off[s] + (size_t)ix * H.np[s] + (size_t)cell];
        };

        // ---- O0: per-p1 setup -------------------------------------------------------------
        const Grid& g1 = H.grid[role.s[0]];
        int i1[3];
        i1[2] = ip1 % g1.n[2]; i1[1] = (ip1 / g1.n[2]) % g1.n[1]; i1[0] = ip1 / (g1.n[2] * g1.n[1]);
        R p1[3];
        for (int d = 0; d < 3; ++d) {
            const R delta = (R)((g1.pmax[d] - g1.pmin[d]) / (double)g1.n[d]);
            p1[d] = rfma<R>((R)i1[d] + (R)0.5, delta, k.pmin[0][d]);
        }
        const R q1 = dot3<R>(p1, p1);
        const R E1 = std::sqrt(q1 + k.msq[0]);
        const R T1 = q1 / (E1 + k.m[0]);        // kinetic energy E1-m1, cancellation-free (float chain)
        const R f1 = fval(0, ip1, p1);
        const R F1 = rfma<R>(k.theta_kappa[0], f1, (R)1);

        for (int n = 0; n < N; ++n) {
            Trace tr; std::memset(&tr, 0, sizeof tr);
            const bool want = trace && n == trace_n;
            // ---- O1/O2: one Philox call per sample; partner momentum uniform in the species-2 box
            // from the top 24 bits of words 0..2; its cell from the same bits by integer arithmetic.
            const U4 r0 = philox4x32_10(key0, key1, (uint32_t)n, (uint32_t)ip1, (uint32_t)ix, (uint32_t)irole);
            R p2[3]; int j2d[3];
            for (int d = 0; d < 3; ++d) {
                const R u = u01<R>(r0.v[d]);
                p2[d] = rfma<R>(u, k.L[1][d], k.pmin[1][d]);
                j2d[d] = (int)(((uint64_t)(r0.v[d] >> 8) * (uint64_t)k.n[1][d]) >> 24);   // = floor(u n)
            }
            const int j2 = (j2d[0] * k.n[1][1] + j2d[1]) * k.n[1][2] + j2d[2];
            // the low bytes of words 0..2 make the 24-bit azimuth index, word 3 gives cos(theta)
            const uint32_t k24 = ((r0.v[0] & 255u) << 16) | ((r0.v[1] & 255u) << 8) | (r0.v[2] & 255u);
            int status = 0, draws = 1;
            R E2 = 0, s = 0, t = 0, u = 0, pf = 0, w = 0, E3 = 0, f2 = 0, f3 = 0, f4 = 0, gain = 0, loss = 0;
            R p3[3] = {0, 0, 0}, p4[3] = {0, 0, 0};
            int j3 = -1, j4 = -1;
            do {
                // ---- O3: partner energy ---------------------------------------------------
                const R q2 = dot3<R>(p2, p2);
                E2 = std::sqrt(q2 + k.msq[1]);
                // ---- O4: s via h = E1 E2 - m1 m2 - p1.p2 = (s - (m1+m2)^2)/2 --------------
                const R d12 = dot3<R>(p1, p2);
                R Kk;
                if (std::is_same<R, float>::value) {
                    // float chain: E1E2 - m1m2 = T1 T2 + m1 T2 + m2 T1 with T = q/(E+m) (no cancellation)
                    const R T2 = q2 / (E2 + k.m[1]);
                    Kk = rfma<R>(T1, T2, rfma<R>(k.m[0], T2, k.m[1] * T1));
                } else {
                    Kk = rfma<R>(E1, E2, -k.m1m2);
                }
                const R h = Kk - d12;
                if (!(h > (R)0)) { status = 1; break; }
                s = rfma<R>((R)2, h, k.msum2);
                const R rs = std::sqrt(s);
                const R irs = (R)1 / rs;
                const R hirs = (R)0.5 * irs;
                // ---- O5: threshold, outgoing CM momentum and CM energy of particle 3 ------
                const R a34 = rfma<R>((R)2, h, k.Mth);          // s - (m3+m4)^2
                if (!(a34 > (R)0)) { status = 2; break; }
                const R b34 = s - k.Mdf;                        // s - (m3-m4)^2
                pf = std::sqrt(a34 * b34) * hirs;               // |p*_34|
                const R E3s = (s + k.dm34) * hirs;              // (s + m3^2 - m4^2) / (2 sqrt s)
                R p3s[3], P[3];
                for (int d = 0; d < 3; ++d) P[d] = p1[d] + p2[d];
                const R Et = E1 + E2;
                const R ig = (R)1 / (Et + rs);
                const R ers = E2 * rs;
                bool weight_done = false;
                if (role.sampler == SAMPLER_TCHANNEL) {
                    // ---- S1: CM momentum of particle 1 (inverse of the boost of O7; E1* = E3* for elastic roles)
                    const R cb = (E1 + E3s) * ig;
                    R v1[3];
                    for (int d = 0; d < 3; ++d) v1[d] = rfma<R>(-P[d], cb, p1[d]);
                    // ---- S2: om = 1 - cos(theta*) from the inverse CDF of 1/(t - mD^2)^2, t = -2 pf^2 om:
                    //      om = 2 mD^2 v / (mD^2 + 4 (1 - v) pf^2),  v uniform in (0,1)
                    const R v = uhalf<R>(r0.v[3]), vb = uhalf<R>(~r0.v[3]);
                    const R q = pf * pf;
                    const R den = rfma<R>((R)4 * vb, q, k.mD2);
                    const R om = (k.twomD2 * v) / den;
                    // ---- S3: polar angle
                    const R st = std::sqrt(om * ((R)2 - om));
                    const R ct = (R)1 - om;
                    // ---- S4: azimuth (same lattice and polynomials as O6)
                    R cphi, sphi;
                    azimuth<R>(k24, cphi, sphi);
                    const R A = st * cphi, B = st * sphi;
                    // ---- S5: frame about v1 (Duff et al. 2017 orthonormal basis, scaled by |v1| = pf):
                    //      pf e1 = (pf - sg x xa, -sg x ya, -sg x),  pf e2 = (-x ya, sg pf - y ya, -y),
                    //      sg = sign(z), xa = x / (sg pf + z), ya = y / (sg pf + z)
                    const R sg = v1[2] >= (R)0 ? (R)1 : (R)-1;
                    const R ia = (R)1 / rfma<R>(sg, pf, v1[2]);
                    const R xa = v1[0] * ia, ya = v1[1] * ia;
                    const R sx = sg * v1[0];
                    const R e1x = rfma<R>(-sx, xa, pf), e1y = -(sx * ya), e1z = -sx;
                    const R e2x = -(v1[0] * ya), e2y = rfma<R>(-v1[1], ya, sg * pf), e2z = -v1[1];
                    p3s[0] = rfma<R>(ct, v1[0], rfma<R>(B, e2x, A * e1x));
                    p3s[1] = rfma<R>(ct, v1[1], rfma<R>(B, e2y, A * e1y));
                    p3s[2] = rfma<R>(ct, v1[2], rfma<R>(B, e2z, A * e1z));
                    // ---- S7: weight = |M|^2 pf / (E2 sqrt s) times the importance ratio
                    //      (1/2) / pdf(om) = D^2 / (mD^2 (mD^2 + 4 pf^2)), D = mD^2 - t: the angular factor cancels
                    t = -((R)2 * q) * om;
                    const R zn = k.mD2 * rfma<R>((R)4, q, k.mD2);
                    if (role.kind == M2_COULOMB_SCREENED) w = (k.par0 * pf) / (zn * ers);
                    else                                  w = ((k.g4 * (s * s)) * pf) / (zn * ers);
                    weight_done = true;
                } else {
                    // ---- O6: direction uniform on the sphere, rejection-free and libm-free ---------
                    R nh[3];
                    direction<R>(r0.v[3], k24, nh);
                    for (int d = 0; d < 3; ++d) p3s[d] = pf * nh[d];
                }
                // ---- O7: boost the CM momentum of particle 3 to the lab ---------------------
                const R dPn = dot3<R>(P, p3s);
                E3 = rfma<R>(Et, E3s, dPn) * irs;               // gamma (E3* + beta.p3*)
                const R c = (E3 + E3s) * ig;                    // p3 = p3* + P (E3+E3*)/(Et+sqrt s)
                for (int d = 0; d < 3; ++d) { p3[d] = rfma<R>(P[d], c, p3s[d]); p4[d] = P[d] - p3[d]; }
                // ---- O8/O9/O12: t = (p1-p3)^2 and the weight as one quotient ---------------
                if (weight_done) {
                } else if (role.kind == M2_CONST) {
                    w = (k.par0 * pf) / ers;
                } else if (role.kind == M2_ISO_DSIGMA) {
                    w = ((k.sig64 * s) * pf) / ers;
                } else {
                    R dl[3];
                    for (int d = 0; d < 3; ++d) dl[d] = p1[d] - p3[d];
                    const R dl2 = dot3<R>(dl, dl);
                    const R dE = E1 - E3;
                    t = rfma<R>(dE, dE, -dl2);
                    if (role.kind >= M2_QCD_Q1Q2) {
                        u = (k.msqsum - s) - t;                 // s + t + u = sum of the squared masses
                        w = (m2_qcd(s, t, u) * pf) / ers;
                    } else {
                        const R D = t - k.mD2;
                        const R den = (D * D) * ers;
                        if (role.kind == M2_COULOMB_SCREENED) w = (k.par0 * pf) / den;
                        else                                  w = ((k.g4 * (s * s)) * pf) / den;
                    }
                }
                // ---- O10: gathers ------------------------------------------------------------
                j3 = cell_of(2, p3); j4 = cell_of(3, p4);
                f2 = fval(1, j2, p2); f3 = fval(2, j3, p3); f4 = fval(3, j4, p4);
                // ---- O11: statistics and integrand (Eq. 16 bracket, Eq. 18) -----------------
                const R F2 = rfma<R>(k.theta_kappa[1], f2, (R)1);
                const R F3 = rfma<R>(k.theta_kappa[2], f3, (R)1);
                const R F4 = rfma<R>(k.theta_kappa[3], f4, (R)1);
                gain = k.cg * ((f3 * f4) * (F1 * F2));
                loss = k.cl * ((f1 * f2) * (F3 * F4));
                // ---- O12: accumulate in double ---------------------------------------------
                const double wg = (double)(w * gain), wl = (double)(w * loss);
                acc.G += wg; acc.Ls += wl;
                // float chain only: the contribution to C is the difference rounded once to float,
                // accumulated in double (O12); the double chain uses G - Ls
                if (std::is_same<R, float>::value) acc.D += (double)(w * gain - w * loss);
                if (j3 >= 0 && j4 >= 0) acc.Lin += wl;
                acc.Q += (wg - wl) * (wg - wl);
                if (sink) {
                    // pref0 = hbar^2 V2 / (16 pi E1 N): the O13 prefactor without the symmetry factor
                    const Grid& g2 = H.grid[role.s[1]];
                    const double V2 = (g2.pmax[0] - g2.pmin[0]) * (g2.pmax[1] - g2.pmin[1]) * (g2.pmax[2] - g2.pmin[2]);
                    const double pref0 = (H.hbar * H.hbar) * V2 / (16.0 * M_PI * (double)E1 * (double)N);
                    const double val = std::is_same<R, float>::value ? (double)(w * gain - w * loss) : wg - wl;
                    const int jc[4] = {ip1, j2, j3, j4};
                    for (int k4 = 0; k4 < 4; ++k4) {
                        if (jc[k4] < 0) continue;                      // left the momentum box: lost from the system
                        const int sk = role.s[k4];
                        const size_t idx = H.sp_off[sk] + (size_t)ix * H.np[sk] + (size_t)jc[k4];
                        const double d = sink->fac[k4] * (pref0 * val);
                        const double m = std::fabs(sink->fac[k4]) * (pref0 * (std::fabs(wg) + std::fabs(wl)));
#pragma omp atomic
                        sink->C[idx] += d;
#pragma omp atomic
                        sink->mag[idx] += m;
                    }
                }
            } while (false);
            if (want) {
                for (int d = 0; d < 3; ++d) { tr.p1[d] = p1[d]; tr.p2[d] = p2[d]; tr.p3[d] = p3[d]; tr.p4[d] = p4[d]; }
                tr.E1 = E1; tr.E2 = E2; tr.E3 = E3; tr.s = s; tr.t = t; tr.pf = pf; tr.w = w;
                tr.f1 = f1; tr.f2 = f2; tr.f3 = f3; tr.f4 = f4; tr.gain = gain; tr.loss = loss; tr.u = u;
                tr.j2 = j2; tr.j3 = j3; tr.j4 = j4; tr.status = status; tr.draws = draws;
                *trace = tr;
            }
        }
        (void)T1;
    }

    // O13: scale.  C_role = hbar^2 sym V2 / (16 pi E1 N) (G - Ls), in double.  hbar^2 is the "hbar^2 c" of Eq. 16
    // with c = 1 (reading R8); the other place hbar enters is nbar of Eq. 18.
    double prefactor(int ip1, int N) const {
        const Grid& g1 = H.grid[role.s[0]];
        int i1[3];
        i1[2] = ip1 % g1.n[2]; i1[1] = (ip1 / g1.n[2]) % g1.n[1]; i1[0] = ip1 / (g1.n[2] * g1.n[1]);
        R p1[3];
        for (int d = 0; d < 3; ++d) {
            const R delta = (R)((g1.pmax[d] - g1.pmin[d]) / (double)g1.n[d]);
            p1[d] = rfma<R>((R)i1[d] + (R)0.5, delta, k.pmin[0][d]);
        }
        const R E1 = std::sqrt(dot3<R>(p1, p1) + k.msq[0]);
        const Grid& g2 = H.grid[role.s[1]];
        const double V2 = (g2.pmax[0] - g2.pmin[0]) * (g2.pmax[1] - g2.pmin[1]) * (g2.pmax[2] - g2.pmin[2]);
        return ((H.hbar * H.hbar) * (role.sym * V2)) / (16.0 * M_PI * (double)E1 * (double)N);
    }
};

template <typename R>
int run_collision(const Handle& H, const double* f, double* C, int N, uint64_t seed, int ix_begin, int ix_end,
                  int ix_stride, double* dG, double* dL, double* dLin, double* dQ, FCallback cb, void* user,
                  int box_cut) {
    // C is zeroed for the spatial cells visited, then roles are added in ascending order (O14).
    for (size_t s = 0; s < H.sp.size(); ++s)
        for (int ix = ix_begin; ix < ix_end; ix += ix_stride)
            for (size_t j = 0; j < H.np[s]; ++j) C[H.sp_off[s] + (size_t)ix * H.np[s] + j] = 0.0;
    for (int ir = 0; ir < (int)H.roles.size(); ++ir) {
        Evaluator<R> ev(H, ir, cb, user, box_cut);
        const int s1 = H.roles[ir].s[0];
        const long np1 = (long)H.np[s1];
        const long ncell = (ix_end - ix_begin + ix_stride - 1) / ix_stride;
        const bool serial = cb != nullptr && cb != orc_builtin_thermal;   // Python callbacks are not thread-safe
#pragma omp parallel for schedule(static) if (!serial)
        for (long idx = 0; idx < ncell * np1; ++idx) {
            const int ix = ix_begin + (int)(idx / np1) * ix_stride;
            const int ip1 = (int)(idx % np1);
            Accum acc;
            ev.eval_p1(f, ix, ip1, N, seed, acc, nullptr, -1);
            const double pref = ev.prefactor(ip1, N);
            C[H.sp_off[s1] + (size_t)ix * np1 + ip1] += pref * (std::is_same<R, float>::value ? acc.D : acc.G - acc.Ls);
            const size_t o = H.role_off[ir] + (size_t)ix * np1 + ip1;
            if (dG) dG[o] = pref * acc.G;
            if (dL) dL[o] = pref * acc.Ls;
            if (dLin) dLin[o] = pref * acc.Lin;
            if (dQ) dQ[o] = pref * pref * acc.Q;
        }
    }
    return 0;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C entry points (ctypes-friendly)
// ---------------------------------------------------------------------------------------------
extern "C" {

void orc_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) {
    const U4 r = philox4x32_10(key[0], key[1], ctr[0], ctr[1], ctr[2], ctr[3]);
    for (int i = 0; i < 4; ++i) out[i] = r.v[i];
}

// O6 alone (pin: tests compare it with numpy's cos/sin): words x[0..3] of one Philox call -> n.
void orc_direction(const uint32_t x[4], int use_float, double out[3]) {
    const uint32_t k24 = ((x[0] & 255u) << 16) | ((x[1] & 255u) << 8) | (x[2] & 255u);
    if (use_float) { float nh[3]; direction<float>(x[3], k24, nh); for (int d = 0; d < 3; ++d) out[d] = nh[d]; }
    else { double nh[3]; direction<double>(x[3], k24, nh); for (int d = 0; d < 3; ++d) out[d] = nh[d]; }
}

// O6 by eye (see direction_by_eye): the same words through the textbook definition and the C library.
void orc_direction_by_eye(const uint32_t x[4], int use_float, double out[3]) {
    const uint32_t k24 = ((x[0] & 255u) << 16) | ((x[1] & 255u) << 8) | (x[2] & 255u);
    if (use_float) direction_by_eye<float>(x[3], k24, out); else direction_by_eye<double>(x[3], k24, out);
}

void* orc_create(int nx, int n_species, const Species* sp, const Grid* grid, int n_process, const Process* pr,
                 double hbar, int use_float) {
    Handle* H = new Handle;
    H->nx = nx; H->hbar = hbar; H->use_float = use_float;
    H->sp.assign(sp, sp + n_species);
    H->grid.assign(grid, grid + n_species);
    size_t off = 0;
    for (int s = 0; s < n_species; ++s) {
        H->sp_off.push_back(off);
        const size_t np = (size_t)grid[s].n[0] * grid[s].n[1] * grid[s].n[2];
        H->np.push_back(np);
        off += (size_t)nx * np;
    }
    // Role expansion (Eq. 16 and Eq. 19).  A role (1,2,3,4) is Eq. 16 with the grid
    // particle d(p) = 1, its partner c(k3) = 2 and the incident pair a(k1), b(k2) = 3, 4: gain f3 f4 F1 F2 from
    // 3+4 -> 1+2, loss f1 f2 F3 F4 from the reverse reaction, both with the same |M|^2 (M_{ab<->cd}).
    // A process written a+b -> c+d therefore contributes
    //   to C_a: role (a,b,c,d)      to C_b: role (b,a,d,c)   (if b != a)
    // and, when it is inelastic ({c,d} != {a,b}), also
    //   to C_c: role (c,d,a,b)      to C_d: role (d,c,b,a)   (if d != c);
    // for an elastic process (c == a, d == b) the second pair would repeat the first.  These permutations keep
    // t = (p1-p3)^2 and u = (p1-p4)^2 equal to the t and u of the process as written.
    // Symmetry factor ("1/2 ... when all incident particles are of the same type"): the incident
    // pair of a role is (3,4), so sym = 1/2 iff species 3 == species 4, else 1; sym >= 0 in the process
    // overrides it for every role of that process.
    // Eq. 16 carries 1/p^0 of the grid particle: a massless species whose grid has a cell centre at
    // p = 0 (odd cell counts on a box symmetric about 0) has no finite collision term there.  Such a problem is
    // refused (reading R14): smallest cell-centre energy E_min = sqrt(Sum_d min_i p_d(i)^2 + m^2), with
    // p_d(i) the centre as O0 computes it, must exceed 1e-6 of the smallest cell width.
    for (int i = 0; i < n_process; ++i) {
        const int idx[4] = {pr[i].a, pr[i].b, pr[i].c, pr[i].d};
        for (int j = 0; j < 4; ++j) {
            if (idx[j] < 0 || idx[j] >= n_species) { delete H; return nullptr; }
            const Grid& g = grid[idx[j]];
            double q = sp[idx[j]].mass * sp[idx[j]].mass, dmin = std::numeric_limits<double>::infinity();
            for (int d = 0; d < 3; ++d) {
                const double delta = (g.pmax[d] - g.pmin[d]) / (double)g.n[d];
                double best = std::numeric_limits<double>::infinity();
                for (int c = 0; c < g.n[d]; ++c) best = std::fmin(best, std::fabs(std::fma((double)c + 0.5, delta, g.pmin[d])));
                q += best * best;
                dmin = std::fmin(dmin, delta);
            }
            if (!(std::sqrt(q) > 1e-6 * dmin)) { delete H; return nullptr; }
        }
    }
    size_t roff = 0;
    for (int i = 0; i < n_process; ++i) {
        const Process& p = pr[i];
        const bool elastic = p.c == p.a && p.d == p.b;
        const bool same_sets = (p.c == p.a && p.d == p.b) || (p.c == p.b && p.d == p.a);
        if (!elastic && same_sets) { delete H; return nullptr; }      // write a+b -> b+a as a+b -> a+b
        if (p.kind < M2_CONST || p.kind > M2_KIND_LAST) { delete H; return nullptr; }
        if (p.sampler != SAMPLER_UNIFORM && p.sampler != SAMPLER_TCHANNEL) { delete H; return nullptr; }
        // the t-channel sampler needs an elastic process of a t-channel kind with a non-zero regulator
        if (p.sampler == SAMPLER_TCHANNEL && !(elastic && (p.kind == M2_COULOMB_SCREENED || p.kind == M2_TCHAN_S2) && p.par[1] != 0.0)) { delete H; return nullptr; }
        Role r; r.kind = p.kind; std::memcpy(r.par, p.par, sizeof r.par); r.process = i; r.sampler = p.sampler;
        r.gab = sp[p.a].g * sp[p.b].g;
        r.sym_override = p.sym;
        // Eq. 19 lists, for every species, the processes it takes part in: C_X receives the process once
        // for every DISTINCT way X appears among its external legs.  The legs are numbered 0 = a, 1 = b (one side of the
        // reaction), 2 = c, 3 = d (the other side).  VIEW[v] is the reaction re-labelled with leg v as the grid particle
        // (slot 1): slot 2 is v's companion on its own side, slots 3 and 4 are the far side taken in the order that keeps
        // (p1 - p3)^2 equal to the t of the process as written (a<->c and b<->d are the t-channel partners).
        static const int VIEW[4][4] = {{0, 1, 2, 3}, {1, 0, 3, 2}, {2, 3, 0, 1}, {3, 2, 1, 0}};
        const int leg_species[4] = {p.a, p.b, p.c, p.d};
        for (int v = 0; v < 4; ++v) {
            const int companion = VIEW[v][1];
            // a view is redundant when it describes the same integral as an earlier one:
            //  - its companion leg has already been viewed and carries the same species (the p2 integral of that view
            //    already runs over every partner of that species);
            //  - it looks from the far side of a reaction that is its own reverse (elastic: gain and loss of the
            //    near-side views are already the two directions of the reaction)
            if (companion < v && leg_species[companion] == leg_species[v]) continue;
            if (v >= 2 && elastic) continue;
            for (int slot = 0; slot < 4; ++slot) r.s[slot] = leg_species[VIEW[v][slot]];
            // 1/2 "when all incident particles are of the same type"; the incident pair of a view is its far side
            const bool identical_pair = r.s[2] == r.s[3];
            r.sym = p.sym >= 0 ? p.sym : (identical_pair ? 0.5 : 1.0);
            H->roles.push_back(r);
            H->role_off.push_back(roff);
            roff += (size_t)nx * H->np[r.s[0]];
        }
    }
    H->role_off.push_back(roff);
    return H;
}

void orc_destroy(void* h) { delete (Handle*)h; }
size_t orc_f_elems(const void* h) { const Handle* H = (const Handle*)h; return H->sp_off.back() + (size_t)H->nx * H->np.back(); }
size_t orc_species_offset(const void* h, int s) { return ((const Handle*)h)->sp_off[s]; }
int orc_n_roles(const void* h) { return (int)((const Handle*)h)->roles.size(); }
size_t orc_detail_elems(const void* h) { return ((const Handle*)h)->role_off.back(); }
size_t orc_role_offset(const void* h, int r) { return ((const Handle*)h)->role_off[r]; }
void orc_role_info(const void* h, int r, int s_out[4], int* kind, double* sym, int* process) {
    const Role& R = ((const Handle*)h)->roles[r];
    for (int i = 0; i < 4; ++i) s_out[i] = R.s[i];
    *kind = R.kind; *sym = R.sym; *process = R.process;
}
int orc_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Full sweep over spatial cells ix_begin, ix_begin+stride, ... < ix_end.  C has orc_f_elems
// doubles (only the visited cells are written).  detail arrays (may be null) have
// orc_detail_elems doubles: scaled gain, loss, in-box loss and the sum of squared per-sample
// contributions (for the Monte Carlo standard error), per (role, ix, p1).
// fcb != null switches to analytic-f mode: every f value comes from fcb(species, p, user);
// box_cut != 0 keeps the "zero outside the momentum box" rule in that mode.
int orc_collision(void* h, const double* f, double* C, int n_samples, uint64_t seed, int ix_begin, int ix_end,
                  int ix_stride, double* dG, double* dL, double* dLin, double* dQ, FCallback fcb, void* user,
                  int box_cut) {
    Handle* H = (Handle*)h;
    if (n_samples <= 0 || ix_begin < 0 || ix_end > H->nx || ix_stride <= 0) return -1;
    if (H->use_float)
        return run_collision<float>(*H, f, C, n_samples, seed, ix_begin, ix_end, ix_stride, dG, dL, dLin, dQ, fcb, user, box_cut);
    return run_collision<double>(*H, f, C, n_samples, seed, ix_begin, ix_end, ix_stride, dG, dL, dLin, dQ, fcb, user, box_cut);
}

// NEXT-3: the conservative ("symmetric") estimator, see SymSink.  C and mag (sum of the absolute deposits, the scale
// of the parity tolerance) have orc_f_elems doubles; the visited spatial cells are overwritten.
// slot_mask (tests only; 15 = the estimator proper): bit k set = deposit for slot k+1; the multiplicity m then counts only
// the (role, slot) pairs in the mask, so that a single-slot mask isolates that slot's estimator of its species' C.
int orc_collision_symmetric(void* h, const double* f, double* C, double* mag, int n_samples, uint64_t seed, int ix_begin,
                            int ix_end, int ix_stride, int slot_mask) {
    Handle* H = (Handle*)h;
    if (n_samples <= 0 || ix_begin < 0 || ix_end > H->nx || ix_stride <= 0) return -1;
    for (size_t s = 0; s < H->sp.size(); ++s)
        for (int ix = ix_begin; ix < ix_end; ix += ix_stride)
            for (size_t j = 0; j < H->np[s]; ++j) { C[H->sp_off[s] + (size_t)ix * H->np[s] + j] = 0.0; mag[H->sp_off[s] + (size_t)ix * H->np[s] + j] = 0.0; }
    // DESIGN.md section 4c.  A sample of a role is one reaction {1, 2} <-> {3, 4} with net rate (gain - loss) as seen by
    // slots 1 and 2; slots 3 and 4 see the opposite sign.  Each of the four slots is, by itself, an unbiased estimator of
    // the collision term of the species in that slot, once (i) divided by that species' momentum-cell volume instead of
    // the grid particle's, (ii) given the identical-particle factor of ITS incident pair, which is the pair across the
    // reaction from the slot, and (iii) averaged with all other (role, slot) estimators of the same species and process.
    // Momentum-cell volume per species:
    std::vector<double> cell_volume(H->sp.size());
    for (size_t sidx = 0; sidx < H->sp.size(); ++sidx) {
        double v = 1.0;
        for (int d = 0; d < 3; ++d) v *= (H->grid[sidx].pmax[d] - H->grid[sidx].pmin[d]) / H->grid[sidx].n[d];
        cell_volume[sidx] = v;
    }
    // (iii) how many (role, slot) estimators each process has per species, counted once over the finished role list
    std::map<std::pair<int, int>, int> estimators;      // (process, species) -> count
    for (const Role& r2 : H->roles)
        for (int slot = 0; slot < 4; ++slot)
            if ((slot_mask >> slot) & 1) ++estimators[std::make_pair(r2.process, r2.s[slot])];
    struct SlotRule { double sign; int across[2]; };    // sign of the slot's net rate; the two slots across the reaction
    static const SlotRule RULE[4] = {{+1.0, {2, 3}}, {+1.0, {2, 3}}, {-1.0, {0, 1}}, {-1.0, {0, 1}}};
    for (int ir = 0; ir < (int)H->roles.size(); ++ir) {
        const Role& role = H->roles[ir];
        SymSink sink; sink.C = C; sink.mag = mag;
        for (int slot = 0; slot < 4; ++slot) {
            sink.fac[slot] = 0.0;
            if (!((slot_mask >> slot) & 1)) continue;
            const int species_here = role.s[slot];
            const bool identical_incident = role.s[RULE[slot].across[0]] == role.s[RULE[slot].across[1]];
            const double pair_factor = role.sym_override >= 0 ? role.sym_override : (identical_incident ? 0.5 : 1.0);
            const double volume_ratio = cell_volume[role.s[0]] / cell_volume[species_here];
            const int count = estimators[std::make_pair(role.process, species_here)];
            sink.fac[slot] = RULE[slot].sign * pair_factor * volume_ratio / (double)count;
        }
        const long np1 = (long)H->np[role.s[0]];
        const long ncell = (ix_end - ix_begin + ix_stride - 1) / ix_stride;
        auto body = [&](auto tag) {
            using R = decltype(tag);
            Evaluator<R> ev(*H, ir, nullptr, nullptr, 1);
#pragma omp parallel for schedule(static)
            for (long idx = 0; idx < ncell * np1; ++idx) {
                const int ix = ix_begin + (int)(idx / np1) * ix_stride;
                Accum acc;
                ev.eval_p1(f, ix, (int)(idx % np1), n_samples, seed, acc, nullptr, -1, &sink);
            }
        };
        if (H->use_float) body(float()); else body(double());
    }
    return 0;
}

// One p1 only (analytic or grid mode): returns scaled G, Ls, Lin, Q for (role, ix, ip1).
int orc_collision_point(void* h, const double* f, int role, int ix, int ip1, int n_samples, uint64_t seed,
                        double out[4], FCallback fcb, void* user, int box_cut) {
    Handle* H = (Handle*)h;
    Accum acc; double pref;
    if (H->use_float) { Evaluator<float> ev(*H, role, fcb, user, box_cut); ev.eval_p1(f, ix, ip1, n_samples, seed, acc, nullptr, -1); pref = ev.prefactor(ip1, n_samples); }
    else { Evaluator<double> ev(*H, role, fcb, user, box_cut); ev.eval_p1(f, ix, ip1, n_samples, seed, acc, nullptr, -1); pref = ev.prefactor(ip1, n_samples); }
    out[0] = pref * acc.G; out[1] = pref * acc.Ls; out[2] = pref * acc.Lin; out[3] = pref * pref * acc.Q;
    return 0;
}

// Kinematics of sample n of (role, ix, ip1): 26 doubles + 5 ints, see struct Trace.
int orc_trace(void* h, const double* f, int role, int ix, int ip1, int n, uint64_t seed, double* dout, int* iout,
              FCallback fcb, void* user, int box_cut) {
    Handle* H = (Handle*)h;
    Trace tr; Accum acc;
    if (H->use_float) { Evaluator<float> ev(*H, role, fcb, user, box_cut); ev.eval_p1(f, ix, ip1, n + 1, seed, acc, &tr, n); }
    else { Evaluator<double> ev(*H, role, fcb, user, box_cut); ev.eval_p1(f, ix, ip1, n + 1, seed, acc, &tr, n); }
    std::memcpy(dout, &tr, 26 * sizeof(double));
    iout[0] = tr.j2; iout[1] = tr.j3; iout[2] = tr.j4; iout[3] = tr.status; iout[4] = tr.draws;
    return 0;
}

// |M|^2(s,t,u) of a Table III role exactly as the sample loop evaluates it (pins: tests/test_oracle_qcd.py).
double orc_m2_qcd(void* h, int role, double s, double t, double u) {
    Handle* H = (Handle*)h;
    if (role < 0 || role >= (int)H->roles.size() || H->roles[role].kind < M2_QCD_Q1Q2) return std::numeric_limits<double>::quiet_NaN();
    Evaluator<double> ev(*H, role, nullptr, nullptr, 1);
    return ev.m2_qcd(s, t, u);
}

// O-update (Eq. 27; positivity PAPER.md:263): f_out = f + dt*C, count f_out < 0.
long orc_update(size_t n, const double* f, const double* C, double dt, double* f_out) {
    long neg = 0;
    for (size_t i = 0; i < n; ++i) { f_out[i] = f[i] + dt * C[i]; if (f_out[i] < 0.0) ++neg; }
    return neg;
}

}  // extern "C"
