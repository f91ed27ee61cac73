// S1c/S1d: right-hand-side construction, per-right-hand-side PCG scalars (device resident, no host
// round trip for alpha/beta), and the port gather.  The solution vector x is never stored: only its
// values at the port nodes (x_port += alpha * p[port]) and its mean are accumulated -- Z_t needs
// nothing else.
#pragma once
#include "common.cuh"

namespace pdn {

// r[b] = e_{node[src[b]]} - 1/n2  (consistent right-hand side of the singular tier system) on the
// pitched plane (plane = ny*pitch doubles; pad entries 0); node[] holds pitched offsets y*pitch + x of the
// tier's ports, src[b] is the port index right-hand side b is the source of.
__global__ void k_init_rhs(double* __restrict__ r, int nx, int pitch, size_t plane, double inv_n2,
                           const int* __restrict__ node, const int* __restrict__ src, int B,
                           const int* __restrict__ skip = nullptr) {
    // two adjacent columns (one 16-byte store) per thread and step; pitch and plane are even
    const int b = blockIdx.y;
    if (skip && skip[b]) return;  // (guess.cuh: this right-hand side starts from its closed-form guess)
    const size_t hot = (size_t)node[src[b]];
    double2* r2 = reinterpret_cast<double2*>(r + b * plane);
    for (size_t i2 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; 2 * i2 < plane; i2 += (size_t)gridDim.x * blockDim.x) {
        const size_t i = 2 * i2;
        const int x = (int)(i % pitch);
        double2 v = make_double2(x < nx ? -inv_n2 : 0.0, x + 1 < nx ? -inv_n2 : 0.0);
        if (i == hot) v.x += 1.0;
        if (i + 1 == hot) v.y += 1.0;
        r2[i2] = v;
    }
}

__global__ void k_pcg_init(PcgScalars s, int B, double bnorm2) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b == 0) *s.n_active = B;
    if (b >= B) return;
    s.rho[b] = 1.0; s.rz[b] = 0.0; s.pq[b] = 0.0; s.rr[b] = 0.0; s.sump[b] = 0.0; s.pap[b] = 0.0; s.psum[b] = 0.0;
    s.alpha[b] = 0.0; s.beta[b] = 0.0; s.xmean[b] = 0.0; s.arho[b] = 0.0; s.qq[b] = 0.0; s.rq[b] = 0.0; s.rrk[b] = bnorm2; s.relres[b] = 1.0; s.active[b] = 1;
}

// After the V-cycle: beta = rz / rho_old (0 on the first iteration or when frozen); rho = rz.
__global__ void k_scal_beta(PcgScalars s, int B, int first) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const double rz = s.rz[b], rho_old = s.rho[b];
    s.beta[b] = (first || !s.active[b] || !(rho_old > 0.0)) ? 0.0 : rz / rho_old;
    s.rho[b] = rz;
    s.rz[b] = 0.0;
    s.pq[b] = 0.0;
    s.sump[b] = 0.0;
    s.qq[b] = 0.0;
    s.rq[b] = 0.0;
}

// After w = L z, q = w + beta q_old (k_pq3).  The direction p = z + beta p_old is implicit:
//   p.Lp   = z.Lz - beta^2 p_old.Lp_old     (p is L-conjugate to p_old, so z.Lp_old = -beta p_old.Lp_old)
//   sum(p) = sum(z) + beta sum(p_old)
// alpha = rho / p.Lp (0 when frozen); xmean += alpha * sum(p) / n2.
__global__ void k_scal_alpha(PcgScalars s, int B, double inv_n2) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b == 0) *s.n_active = 0;  // counted again by k_scal_check
    if (b >= B) return;
    if (!s.active[b]) { s.alpha[b] = 0.0; s.rr[b] = 0.0; return; }  // frozen: nothing of it is maintained any more
    const double bt = s.beta[b];
    const double pap = fma(-bt * bt, s.pap[b], s.pq[b]);
    const double psum = fma(bt, s.psum[b], s.sump[b]);
    s.pap[b] = pap;
    s.psum[b] = psum;
    const double a = pap > 0.0 ? s.rho[b] / pap : 0.0;
    s.alpha[b] = a;
    s.arho[b] = fma(a, s.rho[b], s.arho[b]);
    s.xmean[b] = fma(a * inv_n2, psum, s.xmean[b]);
    s.rr[b] = 0.0;
}

// After k_pq3_last and k_scal_alpha, in place of a pass over r and q:
//   ||r - alpha q||^2 = ||r||^2 - 2 alpha r.q + alpha^2 ||q||^2
// from the sums k_pq3_last left and ||r||^2 of the last check.  The three terms cancel down to the new norm, so the
// rounding error of the sum is bounded by ~1e-13 of their magnitudes (FP64 sums over <= 1e8 nodes); an estimate below
// 100 times that bound is not trusted and the right-hand side is reported as it was (not converged: the host then
// forms the residual itself).
__global__ void k_scal_estimate(PcgScalars s, int B) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B || !s.active[b]) return;
    const double a = s.alpha[b], r0 = s.rrk[b], t1 = 2.0 * a * s.rq[b], t2 = a * a * s.qq[b];
    const double est = (r0 - t1) + t2;
    const double noise = 1e-13 * (r0 + fabs(t1) + t2);
    s.rr[b] = (est > 100.0 * noise) ? est : r0;
}

// After r -= alpha q: convergence test  ||r||^2 <= tol2 * ||b||^2  (||b||^2 = 1 - 1/n2).
__global__ void k_scal_check(PcgScalars s, int B, double tol2, double bnorm2) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    if (s.active[b]) {
        const double rr = s.rr[b];
        s.rrk[b] = rr;
        s.relres[b] = sqrt(rr / bnorm2);
        if (!(rr > tol2 * bnorm2)) s.active[b] = 0;  // also freezes on NaN (reported by the host: PDN_E_NUMERIC)
        else atomicAdd(s.n_active, 1);
    }
}

// Residual update alone, without the V-cycle's down stage -- launched when the batch is expected to converge
// in this iteration, so that the smoothing of a cycle nobody needs is not run:
//   r_out = r_in - alpha q ;  rr += ||r_out||^2      for the right-hand sides still iterating.
// grid = (chunks of the plane, B); 16-byte accesses; plane (= ny*pitch) is even.
constexpr int RESID_THREADS = 256, RESID_PER_THREAD = 8;  // double2 per thread and vector: all loads are issued before the first use
// r_out == nullptr: only the norm (2 V instead of 3 V) -- a batch that is expected to converge now needs its new
// residual only if the expectation fails.
__global__ void __launch_bounds__(RESID_THREADS)
k_resid_update(const double* __restrict__ r_in, const double* __restrict__ q, const double* __restrict__ alpha,
               const int* __restrict__ active, double* __restrict__ r_out, double* __restrict__ rr_acc, size_t plane) {
    __shared__ double red[32];
    const int b = blockIdx.y;
    if (!active[b]) return;
    const double al = alpha[b];
    const size_t n2 = plane / 2, base = (size_t)blockIdx.x * RESID_THREADS * RESID_PER_THREAD + threadIdx.x;
    const double2* r2 = reinterpret_cast<const double2*>(r_in + b * plane);
    const double2* q2 = reinterpret_cast<const double2*>(q + b * plane);
    double2* o2 = r_out ? reinterpret_cast<double2*>(r_out + b * plane) : nullptr;
    double2 rv[RESID_PER_THREAD], qv[RESID_PER_THREAD];
#pragma unroll
    for (int k = 0; k < RESID_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * RESID_THREADS;
        const bool ok = i < n2;
        rv[k] = ok ? __ldcs(r2 + i) : make_double2(0.0, 0.0);  // (streaming: neither vector is read again soon)
        qv[k] = ok ? __ldcs(q2 + i) : make_double2(0.0, 0.0);
    }
    double rr = 0.0;
#pragma unroll
    for (int k = 0; k < RESID_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * RESID_THREADS;
        double2 r = rv[k];
        r.x = fma(-al, qv[k].x, r.x);
        r.y = fma(-al, qv[k].y, r.y);
        if (o2 && i < n2) o2[i] = r;
        rr = fma(r.x, r.x, rr);
        rr = fma(r.y, r.y, rr);
    }
    rr = block_sum(rr, red);
    if (threadIdx.x == 0) atomicAdd(rr_acc + b, rr);
}

// The search direction exists only at the gathered nodes:  pp = z[b][node] + beta[b] * pp  (pp = z on the first
// iteration), then  x_port[b][k] += alpha[b] * pp[b][k],  k over the gather list (all ports of the tier for a
// TSV-source batch; for a terminal batch ngather == 0 and only the source node itself is kept, in pown / xown).
__global__ void k_xport(const double* __restrict__ z, size_t n2, const double* __restrict__ alpha,
                        const double* __restrict__ beta, const int* __restrict__ node, int ngather,
                        const int* __restrict__ src, double* __restrict__ pport, double* __restrict__ pown,
                        double* __restrict__ xport, double* __restrict__ xown, int B, int first) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    const double a = alpha[b];
    if (a == 0.0) return;  // frozen right-hand side: its z is no longer maintained
    const double bt = beta[b];
    if (ngather > 0) {
        if (k < ngather) {
            const size_t i = (size_t)b * ngather + k;
            const double zz = z[b * n2 + node[k]];
            const double pp = first ? zz : fma(bt, pport[i], zz);
            pport[i] = pp;
            xport[i] = fma(a, pp, xport[i]);
        }
    } else if (k == 0) {
        const double zz = z[b * n2 + node[src[b]]];
        const double pp = first ? zz : fma(bt, pown[b], zz);
        pown[b] = pp;
        xown[b] = fma(a, pp, xown[b]);
    }
}

// ZT[src[b]][k] = x_port[b][k] - mean(x_b)   /   zdiag[src[b] - ntsv] = x_own[b] - mean(x_b)
__global__ void k_finish_tsv(const double* __restrict__ xport, const double* __restrict__ xmean, int ngather,
                             const int* __restrict__ src, double* __restrict__ ZT, int B) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    if (k < ngather) ZT[(size_t)src[b] * ngather + k] = xport[(size_t)b * ngather + k] - xmean[b];
}

__global__ void k_finish_term(const double* __restrict__ xown, const double* __restrict__ xmean,
                              const int* __restrict__ src, int ntsv, double* __restrict__ zdiag, int B) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < B) zdiag[src[b] - ntsv] = xown[b] - xmean[b];
}

// TSV re-planning (pdn_update_tsvs): copy the kept entries of a tier's port matrix into its new layout.
//   ZTn[rmap[j]][cmap[k]] = ZTo[j][k]   for old TSV rows j and old ports k whose maps are >= 0
__global__ void k_remap_zt(const double* __restrict__ ZTo, int ntsv_o, int q_o, const int* __restrict__ rmap,
                           const int* __restrict__ cmap, double* __restrict__ ZTn, int q_n) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= q_o) return;
    const int kn = cmap[k];
    for (int j = blockIdx.y; j < ntsv_o; j += gridDim.y) {
        const int jn = rmap[j];
        if (jn >= 0 && kn >= 0) ZTn[(size_t)jn * q_n + kn] = ZTo[(size_t)j * q_o + k];
    }
}

// ... and fill the columns of the added TSV ports in the kept rows by symmetry: Z[j][s] = Z[s][j].
__global__ void k_mirror_added(double* __restrict__ ZT, int ntsv, int q, const int* __restrict__ added, int n_added,
                               const unsigned char* __restrict__ is_added) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n_added) return;
    const int s = added[a];
    for (int j = blockIdx.y; j < ntsv; j += gridDim.y)
        if (!is_added[j]) ZT[(size_t)j * q + s] = ZT[(size_t)s * q + j];
}

// Meshes with n <= 4 are their own coarsest level: Z comes straight from the dense pseudo-inverse.
__global__ void k_direct_small(const double* __restrict__ pinv, int nx, int pitch, int nc,
                               const int* __restrict__ node, int ntsv, int nrows, int q, double* __restrict__ ZT,
                               double* __restrict__ zdiag) {
    const int j = blockIdx.x;
    const int dj = (node[j] / pitch) * nx + node[j] % pitch;
    for (int k = threadIdx.x; k < q; k += blockDim.x) {
        const int dk = (node[k] / pitch) * nx + node[k] % pitch;
        if (j < nrows) ZT[(size_t)j * q + k] = pinv[dj * nc + dk];
        if (j >= ntsv && k == 0) zdiag[j - ntsv] = pinv[dj * nc + dj];
    }
}

// zdiag[s] = ZT[ntsv+s][ntsv+s] when the terminal rows are kept (PDN_TERMINAL_PAIRS)
__global__ void k_zdiag_from_rows(const double* __restrict__ ZT, int q, int ntsv, int nterm, double* __restrict__ zdiag) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < nterm) zdiag[s] = ZT[(size_t)(ntsv + s) * q + ntsv + s];
}

// Coarsest level: e = pinv * r, one thread per (b, i); nc = ny*nx <= 16; vectors are pitched.
__global__ void k_coarse_pinv(const double* __restrict__ pinv, int nx, int pitch, int nc, size_t plane,
                              const double* __restrict__ r, double* __restrict__ e, int B) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= B * nc) return;
    const int b = t / nc, i = t % nc;
    double s = 0.0;
    for (int j = 0; j < nc; ++j) s = fma(__ldg(pinv + i * nc + j), r[b * plane + (j / nx) * pitch + j % nx], s);
    e[b * plane + (i / nx) * pitch + i % nx] = s;
}

}  // namespace pdn
