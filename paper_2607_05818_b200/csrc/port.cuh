// S2 (assembly of the reusable coefficient matrix, Eq. 18), the multiplier part of S3,
// and S4 (pair evaluation, Eq. 22) in the build's Z-notation.
//
// Per tier t the port reduction leaves  ZT_t[j][k] = (L_t^+)[port j, port k]  for the TSV ports j
// (rows, ntsv_t of them) against ALL ports k of the tier (q_t columns), and zdiag_t[s] = (L_t^+)[s,s]
// for the terminal ports (bumps on tier 0, loads on tier d-1).  Port order of tier t:
//   [lower ends of interface t-1] ++ [upper ends of interface t] ++ [terminals].
#pragma once
#include "common.cuh"

namespace pdn {

// Diagonal block K_ii = sym(Z_i[up_i,up_i]) + sym(Z_{i+1}[lo_i,lo_i]) + diag(Rt_i)      (p x p)
//   ZTa = ZT_i (ld qa), up_i ports start at offset oa;  ZTb = ZT_{i+1} (ld qb), lo_i ports start at 0.
__global__ void k_assemble_diag(int p, const double* __restrict__ ZTa, int64_t qa, int oa,
                                const double* __restrict__ ZTb, int64_t qb, const double* __restrict__ rt,
                                double* __restrict__ Kii) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= p) return;
    for (int a = blockIdx.y; a < p; a += gridDim.y) {  // (rows walk gridDim.y, which is capped at 65535)
        double v = 0.5 * (ZTa[(oa + a) * qa + oa + b] + ZTa[(oa + b) * qa + oa + a]) +
                   0.5 * (ZTb[a * qb + b] + ZTb[b * qb + a]);
        if (a == b) v += rt[a];
        Kii[(int64_t)a * p + b] = v;
    }
}

// Coupling block K_{i,i+1} = -sym-part of Z_{i+1}[lo_i, up_{i+1}]          (p_i x p_{i+1})
//   ZT = ZT_{i+1} (ld q); lo_i ports at offset 0, up_{i+1} ports at offset p_i.
__global__ void k_assemble_coupling(int pi, int pj, const double* __restrict__ ZT, int64_t q, double* __restrict__ V) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= pj) return;
    for (int a = blockIdx.y; a < pi; a += gridDim.y) V[(int64_t)a * pj + b] = -0.5 * (ZT[a * q + pi + b] + ZT[(pi + b) * q + a]);
}

// Right-hand-side block row i of F = [F^1 | F^d | B]  (p_i x nrhs, nrhs = m + n + d-1), Eq. (19)/(21):
//   block 0   , cols [0, m)      : Z_0[up_0, bump]       = ZT0[a][ntsv0 + s]
//   block d-2 , cols [m, m+n)    : Z_{d-1}[lo_{d-2}, load] = ZTd[a][ntsvd + l]   (lo ports at offset 0)
//   block i   , col  m+n+i       : 1   (the constraint column 1_{p_i}, Eq. 11)
__global__ void k_assemble_rhs(int i, int dm1, int p, int m, int n, const double* __restrict__ ZT0, int64_t q0,
                               int ntsv0, const double* __restrict__ ZTd, int64_t qd, int ntsvd,
                               double* __restrict__ F) {
    const int nrhs = m + n + dm1;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nrhs) return;
    for (int a = blockIdx.y; a < p; a += gridDim.y) {
        double v = 0.0;
        if (c < m) {
            if (i == 0) v = ZT0[a * q0 + ntsv0 + c];
        } else if (c < m + n) {
            if (i == dm1 - 1) v = ZTd[a * qd + ntsvd + (c - m)];
        } else if (c - m - n == i) {
            v = 1.0;
        }
        F[(int64_t)a * nrhs + c] = v;
    }
}

// G[i][c] = sum over the rows of block i of T_i[a][c]   (= B^T K^-1 F)
__global__ void k_colsum(int p, int nrhs, const double* __restrict__ T, double* __restrict__ Grow) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nrhs) return;
    double s = 0.0;
    for (int a = 0; a < p; ++a) s += T[(int64_t)a * nrhs + c];
    Grow[c] = s;
}

// Multipliers: S = G[:, m+n:] ((d-1)^2, SPD);  Y[i][c] = sum_k Sinv[i][k] (G[k][c] - 1/2) for c < m+n.
// One block; thread 0 inverts S by Gauss-Jordan (d-1 is the number of interfaces, small).
__global__ void k_multipliers(int dm1, int mn, const double* __restrict__ G, double* __restrict__ Sinv,
                              double* __restrict__ Y, int* __restrict__ fail) {
    const int nrhs = mn + dm1;
    if (threadIdx.x == 0) {
        for (int i = 0; i < dm1; ++i)
            for (int j = 0; j < dm1; ++j) Sinv[i * dm1 + j] = (i == j) ? 1.0 : 0.0;
        // work on a copy of S stored behind Sinv
        double* S = Sinv + dm1 * dm1;
        for (int i = 0; i < dm1; ++i)
            for (int j = 0; j < dm1; ++j) S[i * dm1 + j] = G[(int64_t)i * nrhs + mn + j];
        for (int k = 0; k < dm1; ++k) {
            const double piv = S[k * dm1 + k];
            if (!(piv > 0.0)) { *fail = 1; break; }
            const double inv = 1.0 / piv;
            for (int j = 0; j < dm1; ++j) { S[k * dm1 + j] *= inv; Sinv[k * dm1 + j] *= inv; }
            for (int i = 0; i < dm1; ++i) {
                if (i == k) continue;
                const double f = S[i * dm1 + k];
                if (f == 0.0) continue;
                for (int j = 0; j < dm1; ++j) {
                    S[i * dm1 + j] -= f * S[k * dm1 + j];
                    Sinv[i * dm1 + j] -= f * Sinv[k * dm1 + j];
                }
            }
        }
    }
    __syncthreads();
    for (int c = threadIdx.x; c < mn; c += blockDim.x)
        for (int i = 0; i < dm1; ++i) {
            double s = 0.0;
            for (int k = 0; k < dm1; ++k) s = fma(Sinv[i * dm1 + k], G[(int64_t)k * nrhs + c] - 0.5, s);
            Y[(int64_t)i * mn + c] = s;
        }
}

// TSV currents of block row i:  I[a][c] = T[a][c] - sum_k T[a][m+n+k] Y[k][c]   for c < m+n  (in place)
__global__ void k_currents(int p, int dm1, int mn, double* __restrict__ T, const double* __restrict__ Y) {
    const int nrhs = mn + dm1;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= mn) return;
    for (int a = blockIdx.y; a < p; a += gridDim.y) {
        double v = T[(int64_t)a * nrhs + c];
        for (int k = 0; k < dm1; ++k) v = fma(-T[(int64_t)a * nrhs + mn + k], Y[(int64_t)k * mn + c], v);
        T[(int64_t)a * nrhs + c] = v;
    }
}

// Terminal constants (one thread per terminal column c of the first / last block row):
//   s = zdiag[c] - ( sum_a f[a][c] I[a][c] + 1/2 sum_k Y[k][col] )  [ - sum_k Y[k][col]  for loads ]
// f[a][c] = ZT[a*q + ntsv + c] (original right-hand side), I = solved block row (ld nrhs, column col0 + c).
__global__ void k_terminal_consts(int p, int dm1, int mn, int nterm, int col0, int is_load,
                                  const double* __restrict__ ZT, int64_t q, int ntsv, int row_off,
                                  const double* __restrict__ I, const double* __restrict__ Y,
                                  const double* __restrict__ zdiag, double* __restrict__ out) {
    const int nrhs = mn + dm1;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nterm) return;
    double s = 0.0;
    for (int a = 0; a < p; ++a) s = fma(ZT[(int64_t)(row_off + a) * q + ntsv + c], I[(int64_t)a * nrhs + col0 + c], s);
    double ys = 0.0;
    for (int k = 0; k < dm1; ++k) ys += Y[(int64_t)k * mn + col0 + c];
    out[c] = zdiag[c] - (s + 0.5 * ys) - (is_load ? ys : 0.0);
}

// Packed operands of the pair kernel:  A1[s][a] = Z_0[up_0 a, bump s]  (m x p0);
//                                      X0[l][a] = I_{load l}[block 0, a]  (n x p0).
__global__ void k_pack_pair_operands(int p0, int m, int n, int dm1, const double* __restrict__ ZT0, int64_t q0,
                                     int ntsv0, const double* __restrict__ I0, double* __restrict__ A1,
                                     double* __restrict__ X0) {
    const int nrhs = m + n + dm1;
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= p0) return;
    for (int row = blockIdx.y; row < m + n; row += gridDim.y) {
        if (row < m) A1[(int64_t)row * p0 + a] = ZT0[(int64_t)a * q0 + ntsv0 + row];
        else X0[(int64_t)(row - m) * p0 + a] = I0[(int64_t)a * nrhs + m + (row - m)];
    }
}

// Same-side pairs (Eq. (4) PAPER.md:60-65 needs the load-load ones).  For two terminals
// i, j of the same tier the unit current enters and leaves on that tier, b = b_i - b_j carries no net current
// through any interface (the constraint entries cancel), and with x_i = C^-1 b_i (already solved for every
// terminal in S3)
//     R(i,j) = t_i + t_j - 2 ( Z[i,j] - b_i^T x_j ),   t_i = Z[i,i] - b_i^T x_i,
//     b_i^T x_j = sum_a A[i][a] X[j][a] + ys[j],
// A[i][a] = Z_t[tsv port a, terminal i] over the p ports of the adjacent interface, X[j][a] = that block of
// the currents of x_j, ys[j] = 1/2 sum_k y_j[k].
__global__ void k_pack_side(int p, int nt, int col0, int nrhs, const double* __restrict__ ZT, int64_t q, int ntsv,
                            const double* __restrict__ Iblk, double* __restrict__ A, double* __restrict__ X) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= p) return;
    for (int s = blockIdx.y; s < nt; s += gridDim.y) {
        A[(int64_t)s * p + a] = ZT[(int64_t)a * q + ntsv + s];
        X[(int64_t)s * p + a] = Iblk[(int64_t)a * nrhs + col0 + s];
    }
}

__global__ void k_side_consts(int p, int nt, int col0, int dm1, int mn, const double* __restrict__ A,
                              const double* __restrict__ X, const double* __restrict__ Y,
                              const double* __restrict__ zdiag, double* __restrict__ ys, double* __restrict__ t) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nt) return;
    double dot = 0.0, y = 0.0;
    for (int a = 0; a < p; ++a) dot = fma(A[(int64_t)s * p + a], X[(int64_t)s * p + a], dot);
    for (int k = 0; k < dm1; ++k) y += Y[(int64_t)k * mn + col0 + s];
    ys[s] = 0.5 * y;
    t[s] = zdiag[s] - (dot + 0.5 * y);
}

// R[i][j] for all ordered pairs of the nt terminals of one side; 64x64 tile / block like k_pair_full.
// ZTT = the terminal rows of the tier's port matrix (row ntsv+i, column ntsv+j), leading dimension q.
__global__ void __launch_bounds__(256)
k_pair_same(int nt, int p, const double* __restrict__ A, const double* __restrict__ X, const double* __restrict__ ys,
            const double* __restrict__ t, const double* __restrict__ ZT, int64_t q, int ntsv, double* __restrict__ R) {
    __shared__ double As[16][65];
    __shared__ double Bs[16][65];
    const int tid = threadIdx.x, tx = tid % 16, ty = tid / 16;
    const int i0 = blockIdx.y * 64, j0 = blockIdx.x * 64;
    double acc[4][4] = {};
    for (int k0 = 0; k0 < p; k0 += 16) {
        for (int e = tid; e < 16 * 64; e += 256) {
            const int kk = e % 16, ii = e / 16;
            As[kk][ii] = (i0 + ii < nt && k0 + kk < p) ? A[(int64_t)(i0 + ii) * p + k0 + kk] : 0.0;
            Bs[kk][ii] = (j0 + ii < nt && k0 + kk < p) ? X[(int64_t)(j0 + ii) * p + k0 + kk] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) a[r] = As[kk][ty * 4 + r];
#pragma unroll
            for (int c = 0; c < 4; ++c) b[c] = Bs[kk][tx + 16 * c];
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[r][c] = fma(a[r], b[c], acc[r][c]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int i = i0 + ty * 4 + r;
        if (i >= nt) continue;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int j = j0 + tx + 16 * c;
            if (j >= nt) continue;
            const double z = 0.5 * (ZT[(int64_t)(ntsv + i) * q + ntsv + j] + ZT[(int64_t)(ntsv + j) * q + ntsv + i]);
            R[(int64_t)i * nt + j] = (i == j) ? 0.0 : (t[i] + t[j]) - 2.0 * (z - (acc[r][c] + ys[j]));
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Arbitrary-tier endpoints (pdn_reff_nodes).  A unit current entering at probe a (tier t_a) is the right-hand
// side  b_a = [f_a; c_a]  of C:  f_a = +Z_t[up_t, a] in block row t (t < d-1), -Z_t[lo_{t-1}, a] in block row
// t-1 (t > 0), zero elsewhere (the KVL rows of Eq. (9)/(16) with the source on tier t), and  c_a[i] = 1 for
// the interfaces i >= t_a below it (the KCL rows, Eq. (11)).  With
//     M = Zloc - [F; Cs]^T C^-1 [F; Cs],     Zloc[a][b] = Z_t[a, b] if t_a = t_b else 0,
// the effective resistance of any pair is  R(a,b) = M_aa + M_bb - M_ab - M_ba  (a constant shift of every c_a,
// e.g. the 1/2 of Eq. (19)/(21), cancels in the difference).
//
// Scatter of one tier's probe rows.  Zp = port matrix of [tsv ports of the tier] ++ [its k probes] (ld q =
// ntsv + k, probe rows ntsv..q-1 valid); probe[j] = column of probe j in the n_nodes-wide arrays; plo = number
// of lower ends (interface t-1) heading the port list.  Fup / Flo = block rows t / t-1 of F (null if absent).
__global__ void k_probe_scatter(int k, int ntsv, int plo, int np, const int* __restrict__ probe,
                                const double* __restrict__ Zp, double* __restrict__ Fup, double* __restrict__ Flo,
                                double* __restrict__ M) {
    const int col = blockIdx.x * blockDim.x + threadIdx.x, q = ntsv + k;
    if (col >= q) return;
    for (int j = blockIdx.y; j < k; j += gridDim.y) {
        const double* row = Zp + (int64_t)(ntsv + j) * q;
        const int a = probe[j];
        if (col < plo) {
            if (Flo) Flo[(int64_t)col * np + a] = -row[col];
        } else if (col < ntsv) {
            if (Fup) Fup[(int64_t)(col - plo) * np + a] = row[col];
        } else {
            const int j2 = col - ntsv;
            M[(int64_t)a * np + probe[j2]] = 0.5 * (row[col] + Zp[(int64_t)(ntsv + j2) * q + ntsv + j]);
        }
    }
}

// Multipliers of the probe right-hand sides:  Cs[i][a] = (tier[a] <= i),  mu[i][a] = sum_k Sinv[i][k] (G[k][a] - Cs[k][a])
__global__ void k_probe_multipliers(int dm1, int np, const double* __restrict__ G, const double* __restrict__ Sinv,
                                    const int* __restrict__ tier, double* __restrict__ Cs, double* __restrict__ mu) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= np) return;
    const int t = tier[a];
    for (int i = 0; i < dm1; ++i) {
        double s = 0.0;
        for (int k = 0; k < dm1; ++k) s = fma(Sinv[i * dm1 + k], G[(int64_t)k * np + a] - (t <= k ? 1.0 : 0.0), s);
        mu[(int64_t)i * np + a] = s;
        Cs[(int64_t)i * np + a] = t <= i ? 1.0 : 0.0;
    }
}

__global__ void k_probe_pairs(int np, const double* __restrict__ M, double* __restrict__ R) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= np) return;
    for (int a = blockIdx.y; a < np; a += gridDim.y)
        R[(int64_t)a * np + b] = a == b ? 0.0 : (M[(int64_t)a * np + a] + M[(int64_t)b * np + b]) - (M[(int64_t)a * np + b] + M[(int64_t)b * np + a]);
}

// One source against many probes (pdn_reff_from): only the row M[s][.] and the diagonal of M are needed, so the
// probe columns of Z_t at the TSV ports come from the TSV-SOURCE solves gathered at the probes (reciprocity,
// Z_t[tsv, a] = x_tsv[a]) and every probe costs only a diagonal (second-order, loosely converged) solve.
//   Zp: rows = the tier's TSV ports [+ the source if it sits on this tier] (nrow of them), columns = [those rows'
//   ports] ++ [the other probes] (q = nrow + k); zd[j] = Z_t[a_j, a_j] of the other probes; col[j] = column of probe j
//   in Zp, probe[j] = its column in the np-wide arrays; src_row = row of the source in Zp or -1.
__global__ void k_from_scatter(int nprobe, int ntsv, int nrow, int plo, int np, int src_row, const int* __restrict__ col,
                               const int* __restrict__ probe, const double* __restrict__ Zp, int64_t q,
                               const double* __restrict__ zd, double* __restrict__ Fup, double* __restrict__ Flo,
                               double* __restrict__ Zd, double* __restrict__ Zs) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    for (int j = blockIdx.y; j < nprobe; j += gridDim.y) {
        const int c = col[j], a = probe[j];
        if (r < ntsv) {
            const double v = Zp[(int64_t)r * q + c];
            if (r < plo) { if (Flo) Flo[(int64_t)r * np + a] = -v; }
            else if (Fup) Fup[(int64_t)(r - plo) * np + a] = v;
        } else if (r == ntsv) {
            Zd[a] = c < nrow ? Zp[(int64_t)c * q + c] : zd[c - nrow];
            Zs[a] = src_row >= 0 ? Zp[(int64_t)src_row * q + c] : 0.0;
        }
    }
}

// qd[a] += sum_r F[r][a] X[r][a],  qs[a] += sum_r F[r][0] X[r][a]   (one interface block; column 0 is the source)
__global__ void k_from_dots(int p, int np, const double* __restrict__ F, const double* __restrict__ X,
                            double* __restrict__ qd, double* __restrict__ qs) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= np) return;
    double d = 0.0, s = 0.0;
    for (int r = 0; r < p; ++r) {
        const double x = X[(int64_t)r * np + a];
        d = fma(F[(int64_t)r * np + a], x, d);
        s = fma(F[(int64_t)r * np], x, s);
    }
    qd[a] += d;
    qs[a] += s;
}

// R(s, a) = M_ss + M_aa - 2 M_sa,  M_ab = Zloc_ab - (F_a . X_b + Cs_a . mu_b);  out[a - 1] for the probes a >= 1
__global__ void k_from_finish(int dm1, int np, const double* __restrict__ Cs, const double* __restrict__ mu,
                              const double* __restrict__ Zd, const double* __restrict__ Zs, const double* __restrict__ qd,
                              const double* __restrict__ qs, double* __restrict__ out) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a < 1 || a >= np) return;
    double cd = 0.0, cs = 0.0, c0 = 0.0;
    for (int i = 0; i < dm1; ++i) {
        cd = fma(Cs[(int64_t)i * np + a], mu[(int64_t)i * np + a], cd);
        cs = fma(Cs[(int64_t)i * np], mu[(int64_t)i * np + a], cs);
        c0 = fma(Cs[(int64_t)i * np], mu[(int64_t)i * np], c0);
    }
    const double mss = Zd[0] - (qd[0] + c0), maa = Zd[a] - (qd[a] + cd), msa = Zs[a] - (qs[a] + cs);
    out[a - 1] = (mss + maa) - 2.0 * msa;
}

// Eq. (4): with bump b at v_bump and load k drawing I[k],
//   v[j] = v_bump - 1/2 sum_k I[k] ( R_b[j] + R_b[k] - R_LL[j][k] )       one warp per load j
__global__ void k_load_voltages(int n, const double* __restrict__ Rb, const double* __restrict__ RLL,
                                const double* __restrict__ I, double v_bump, double* __restrict__ v) {
    const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (j >= n) return;
    double s = 0.0;
    const double rbj = Rb[j];
    for (int k = lane; k < n; k += 32) s = fma(I[k], (rbj + Rb[k]) - RLL[(int64_t)j * n + k], s);
    s = warp_sum(s);
    if (lane == 0) v[j] = v_bump - 0.5 * s;
}

// Single tier (d = 1, a 2-D PDN: no TSVs, nothing to recombine).  The bumps are the row sources of the tier's port
// matrix (ports = [bumps] ++ [loads], ntsv = m), and R(i,j) = Z[b_i,b_i] + Z[l_j,l_j] - 2 Z[b_i,l_j] is Eq. (2) on
// the one mesh.  Written as operands of the pair kernels:  A1 = I (m x m, set by the caller),
// X0[j][a] = Z[b_a, l_j],  u[i] = Z[b_i, b_i],  w[j] = zdiag[j].
__global__ void k_single_tier_operands(int m, int n, const double* __restrict__ ZT, int64_t q,
                                       const double* __restrict__ zdiag, double* __restrict__ X0,
                                       double* __restrict__ u, double* __restrict__ w) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= m) return;
    for (int j = blockIdx.y; j <= n; j += gridDim.y) {
        if (j < n) X0[(int64_t)j * m + a] = ZT[(int64_t)a * q + m + j];
        else u[a] = ZT[(int64_t)a * q + a];
        if (j < n && a == 0) w[j] = zdiag[j];
    }
}

// S4, full cross product:  R[i][j] = u[i] + w[j] - 2 sum_a A1[i][a] X0[j][a].   64x64 tile / block.
__global__ void __launch_bounds__(256)
k_pair_full(int m, int n, int p0, const double* __restrict__ A1, const double* __restrict__ X0,
            const double* __restrict__ u, const double* __restrict__ w, double* __restrict__ R) {
    __shared__ double As[16][65];
    __shared__ double Bs[16][65];
    const int tid = threadIdx.x, tx = tid % 16, ty = tid / 16;
    const int i0 = blockIdx.y * 64, j0 = blockIdx.x * 64;
    double acc[4][4] = {};
    for (int k0 = 0; k0 < p0; k0 += 16) {
        for (int e = tid; e < 16 * 64; e += 256) {
            const int kk = e % 16, ii = e / 16;
            As[kk][ii] = (i0 + ii < m && k0 + kk < p0) ? A1[(int64_t)(i0 + ii) * p0 + k0 + kk] : 0.0;
            Bs[kk][ii] = (j0 + ii < n && k0 + kk < p0) ? X0[(int64_t)(j0 + ii) * p0 + k0 + kk] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) a[r] = As[kk][ty * 4 + r];
#pragma unroll
            for (int c = 0; c < 4; ++c) b[c] = Bs[kk][tx + 16 * c];
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[r][c] = fma(a[r], b[c], acc[r][c]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int i = i0 + ty * 4 + r;
        if (i >= m) continue;
        const double ui = u[i];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int j = j0 + tx + 16 * c;
            if (j < n) R[(int64_t)i * n + j] = ui + w[j] - 2.0 * acc[r][c];
        }
    }
}

// S4, pair list: one warp per pair.
__global__ void k_pair_list(int64_t npairs, int m, int n, int p0, const int* __restrict__ bi,
                            const int* __restrict__ li, const double* __restrict__ A1,
                            const double* __restrict__ X0, const double* __restrict__ u,
                            const double* __restrict__ w, double* __restrict__ R) {
    const int64_t pair = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (pair >= npairs) return;
    const int i = bi[pair], j = li[pair];
    if (i < 0 || i >= m || j < 0 || j >= n) {
        if (lane == 0) R[pair] = nan("");
        return;
    }
    double s = 0.0;
    for (int a = lane; a < p0; a += 32) s = fma(A1[(int64_t)i * p0 + a], X0[(int64_t)j * p0 + a], s);
    s = warp_sum(s);
    if (lane == 0) R[pair] = u[i] + w[j] - 2.0 * s;
}

}  // namespace pdn
