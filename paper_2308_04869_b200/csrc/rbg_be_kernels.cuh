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
// Moments.  One CTA per (species, spatial cell).  Momentum integrals are midpoint sums, Int d3p -> Sum dp^3.
// With g = f / E and q = |p|^2 + m^2 (so E f = q g):
//   n = S f, T^{0k} = S p_k f, j^k = S p_k g, T^{ik} = S p_i p_k g, T^{00} = S q g.
// A lane owns columns of fixed (ipy, ipz) and walks along ipx, so that only five running sums need the per-cell
// arithmetic (X0 = S_x f, X1 = S_x px f, G0 = S_x g, G1 = S_x px g, G2 = S_x px^2 g); the p_y, p_z factors are applied
// once per column.  Loads are coalesced across the lanes of a warp (consecutive (ipy, ipz)).
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
moments_kernel(const double* __restrict__ f_species, SpeciesTables tb, int nx_cells, double* __restrict__ M_species) {
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
        const double py = fma((double)iy + 0.5, tb.delta[1], tb.pmin[1]);
        const double pz = fma((double)iz + 0.5, tb.delta[2], tb.pmin[2]);
        double X0 = 0.0, X1 = 0.0, G0 = 0.0, G1 = 0.0, G2 = 0.0;
#pragma unroll 4
        for (int i = 0; i < tb.n[0]; ++i) {
            const double px = fma((double)i + 0.5, tb.delta[0], tb.pmin[0]);
            const size_t j = (size_t)i * nyz + c;
            const double a = __ldcs(f + j);              // streamed once
            const double g = a * __ldg(iE + j);          // table shared by every spatial cell: L2-resident
            const double pg = px * g;
            X0 += a;
            X1 = fma(px, a, X1);
            G0 += g;
            G1 += pg;
            G2 = fma(px, pg, G2);
        }
        const double r = fma(py, py, fma(pz, pz, msq));                   // q - px^2
        const double yG0 = py * G0, zG0 = pz * G0;
        acc[0] += X0;                                                     // n
        acc[1] += G1; acc[2] += yG0; acc[3] += zG0;                       // j
        acc[4] += fma(r, G0, G2);                                         // T00 = S (px^2 + r) g
        acc[5] += X1; acc[6] = fma(py, X0, acc[6]); acc[7] = fma(pz, X0, acc[7]);   // T0k
        acc[8] += G2; acc[9] = fma(py, G1, acc[9]); acc[10] = fma(pz, G1, acc[10]); // Txx Txy Txz
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
        const double dp3 = tb.delta[0] * tb.delta[1] * tb.delta[2];
        M_species[(size_t)ix * N_MOMENTS + threadIdx.x] = v * dp3;
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
    int slab;                // spatial cells per CTA
};

__global__ void __launch_bounds__(256)
drift_upfd_kernel(const double* __restrict__ f_species, double* __restrict__ out_species, SpeciesTables tb, DriftParams dp) {
    const int nchunks = (tb.np + blockDim.x - 1) / blockDim.x;
    const int chunk = blockIdx.x % nchunks, slab = blockIdx.x / nchunks;
    const int ip = chunk * blockDim.x + threadIdx.x;
    if (ip >= tb.np) return;
    const int nx_cells = dp.nxyz[0] * dp.nxyz[1] * dp.nxyz[2];
    const int ix_begin = slab * dp.slab, ix_end = min(ix_begin + dp.slab, nx_cells);
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
    const int stride[3] = {dp.nxyz[1] * dp.nxyz[2], dp.nxyz[2], 1};
    int i[3];
    i[0] = ix_begin / stride[0]; i[1] = (ix_begin - i[0] * stride[0]) / stride[1]; i[2] = ix_begin - i[0] * stride[0] - i[1] * stride[1];
    for (int ix = ix_begin; ix < ix_end; ++ix) {
        const double* __restrict__ row = f_species + (size_t)ix * tb.np;
        const double self = __ldg(row + ip);
        double num = self * (1.0 / 3.0);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            int j = i[d] - sgn[d];                           // upwind neighbour along d
            double up;
            if ((unsigned)j < (unsigned)dp.nxyz[d]) {
                up = __ldg(row + (ptrdiff_t)(-sgn[d] * stride[d]) * tb.np + ip);
            } else if (dp.bc[d] == 1) {
                j = j < 0 ? dp.nxyz[d] - 1 : 0;
                up = __ldg(row + (ptrdiff_t)((j - i[d]) * stride[d]) * tb.np + ip);
            } else {
                up = dp.zeta != 0.0 ? dp.zeta * __ldg(row + mir[d]) : 0.0;
            }
            num = fma(c[d], up, num);
        }
        out_species[(size_t)ix * tb.np + ip] = num * rden;
        if (++i[2] == dp.nxyz[2]) { i[2] = 0; if (++i[1] == dp.nxyz[1]) { i[1] = 0; ++i[0]; } }
    }
}

struct VlasovParams {
    double dt;
    int nx_cells;
    int slab;
    const double* E;         // [nx_cells][3]
    const double* B;         // [nx_cells][3]
};

__global__ void __launch_bounds__(256)
vlasov_upfd_kernel(const double* __restrict__ f_species, double* __restrict__ out_species, SpeciesTables tb, VlasovParams vp) {
    const int nchunks = (tb.np + blockDim.x - 1) / blockDim.x;
    const int chunk = blockIdx.x % nchunks, slab = blockIdx.x / nchunks;
    const int ip = chunk * blockDim.x + threadIdx.x;
    if (ip >= tb.np) return;
    const int ix_begin = slab * vp.slab, ix_end = min(ix_begin + vp.slab, vp.nx_cells);
    // momentum neighbours of this cell, periodic: [d][0] at p_d - dp_d, [d][1] at p_d + dp_d
    int nb[3][2];        // indexed with compile-time constants only (registers)
    {
        const int nyz = tb.n[1] * tb.n[2];
        const int i0 = ip / nyz, i1 = (ip - i0 * nyz) / tb.n[2], i2 = ip - i0 * nyz - i1 * tb.n[2];
        nb[0][0] = ip + (i0 > 0 ? -nyz : (tb.n[0] - 1) * nyz);
        nb[0][1] = ip + (i0 < tb.n[0] - 1 ? nyz : -(tb.n[0] - 1) * nyz);
        nb[1][0] = ip + (i1 > 0 ? -tb.n[2] : (tb.n[1] - 1) * tb.n[2]);
        nb[1][1] = ip + (i1 < tb.n[1] - 1 ? tb.n[2] : -(tb.n[1] - 1) * tb.n[2]);
        nb[2][0] = ip + (i2 > 0 ? -1 : tb.n[2] - 1);
        nb[2][1] = ip + (i2 < tb.n[2] - 1 ? 1 : -(tb.n[2] - 1));
    }
    const double vx = __ldg(tb.v + ip), vy = __ldg(tb.v + (size_t)tb.np + ip), vz = __ldg(tb.v + 2 * (size_t)tb.np + ip);
    const double k0 = vp.dt / tb.delta[0], k1 = vp.dt / tb.delta[1], k2 = vp.dt / tb.delta[2];
    const double Q = tb.charge;
    for (int ix = ix_begin; ix < ix_end; ++ix) {
        const double* __restrict__ row = f_species + (size_t)ix * tb.np;
        const double* __restrict__ Ev = vp.E + (size_t)ix * 3;
        const double* __restrict__ Bv = vp.B + (size_t)ix * 3;
        const double Ex = __ldg(Ev), Ey = __ldg(Ev + 1), Ez = __ldg(Ev + 2);
        const double Bx = __ldg(Bv), By = __ldg(Bv + 1), Bz = __ldg(Bv + 2);
        // F = Q (E + v x B)
        const double Fx = Q * (Ex + (vy * Bz - vz * By));
        const double Fy = Q * (Ey + (vz * Bx - vx * Bz));
        const double Fz = Q * (Ez + (vx * By - vy * Bx));
        const double c0 = fabs(Fx) * k0, c1 = fabs(Fy) * k1, c2 = fabs(Fz) * k2;
        const double self = __ldg(row + ip);
        const double u0 = __ldg(row + (Fx > 0.0 ? nb[0][0] : nb[0][1]));
        const double u1 = __ldg(row + (Fy > 0.0 ? nb[1][0] : nb[1][1]));
        const double u2 = __ldg(row + (Fz > 0.0 ? nb[2][0] : nb[2][1]));
        const double num = fma(c2, u2, fma(c1, u1, fma(c0, u0, self * (1.0 / 3.0))));
        const double den = ((1.0 / 3.0 + c0) + c1) + c2;
        out_species[(size_t)ix * tb.np + ip] = num / den;
    }
}

}  // namespace rbg
