// Host-side orchestration of S2 + S3: drivers of the dense kernels and the recombination.  Included by
// pdn_api.cu only (after host_solve.cuh).
#pragma once

namespace {

// ------------------------------------------------------------------------------------------------
// ------------------------------------------------------------------------------------------------
// S3 host drivers of the dense kernels (row-major, in place).
void gemm(Launcher& L, int M, int N, int K, double alpha, const double* A, int64_t sai, int64_t sak, const double* B,
          int64_t sbk, int64_t sbj, double beta, double* C, int64_t ldc) {
    if (M <= 0 || N <= 0) return;
    if (M >= 96 && N >= 96 && K >= 16) {  // large enough for the 128x128 tensor-core tiles to pay
        dim3 grid(cdiv(N, DG_BN), cdiv(M, DG_BM));
        L.run(KC_DENSE, 0, [&] { k_gemm_dmma<<<grid, DG_THREADS, 0, L.s>>>(M, N, K, alpha, A, sai, sak, B, sbk, sbj, beta, C, ldc); });
        return;
    }
    dim3 grid(cdiv(N, GEMM_BN), cdiv(M, GEMM_BM));
    L.run(KC_DENSE, 0, [&] { k_gemm<<<grid, 256, 0, L.s>>>(M, N, K, alpha, A, sai, sak, B, sbk, sbj, beta, C, ldc); });
}

// A (n x n, lda) <- its lower Cholesky factor (strict upper part of the diagonal panels zeroed).
void potrf(Launcher& L, double* A, int64_t lda, int n, int* fail) {
    for (int k0 = 0; k0 < n; k0 += DENSE_NB) {
        const int nb = std::min(DENSE_NB, n - k0);
        L.run(KC_DENSE, 0, [&] { k_potrf_diag<<<1, DENSE_NB * DENSE_NB, 0, L.s>>>(A, lda, k0, nb, fail); });
        const int rest = n - k0 - nb;
        if (rest <= 0) break;
        L.run(KC_DENSE, 0, [&] { k_potrf_panel<<<cdiv(rest, 128), 128, 0, L.s>>>(A, lda, n, k0, nb); });
        const double* P = A + (int64_t)(k0 + nb) * lda + k0;  // panel rows (rest x nb)
        gemm(L, rest, rest, nb, -1.0, P, lda, 1, P, 1, lda, 1.0, A + (int64_t)(k0 + nb) * lda + k0 + nb, lda);
    }
}

// Bm (n x nrhs, ldb) <- Lm^-1 Bm
void trsm_fwd(Launcher& L, const double* Lm, int64_t lda, int n, double* Bm, int64_t ldb, int nrhs) {
    for (int k0 = 0; k0 < n; k0 += DENSE_NB) {
        const int nb = std::min(DENSE_NB, n - k0);
        L.run(KC_DENSE, 0, [&] { k_trsm_fwd_diag<<<cdiv(nrhs, 128), 128, 0, L.s>>>(Lm, lda, k0, nb, Bm, ldb, nrhs); });
        const int rest = n - k0 - nb;
        if (rest > 0)
            gemm(L, rest, nrhs, nb, -1.0, Lm + (int64_t)(k0 + nb) * lda + k0, lda, 1, Bm + (int64_t)k0 * ldb, ldb, 1, 1.0,
                 Bm + (int64_t)(k0 + nb) * ldb, ldb);
    }
}

// ------------------------------------------------------------------------------------------------
// F_i <- (K^-1 F)_i for the block rows F_i (p_i x nrhs) of any right-hand-side set, with the factor kept in the
// context (c->Li[i] = L_i^-1, c->Vf[i] = L_{i-1}^-1 K_{i-1,i}): forward then backward block substitution, every
// step a contraction on the FP64 tensor cores.
void block_substitute(pdn_ctx* c, Launcher& L, std::vector<DevBuf>& F, int nrhs) {
    const int dm1 = c->d - 1;
    DevBuf tmp;
    size_t tmax = 0;
    for (int i = 0; i < dm1; ++i) tmax = std::max(tmax, (size_t)c->p[i] * nrhs);
    tmp.alloc(tmax * sizeof(double));
    for (int i = 0; i < dm1; ++i) {
        const int pi = c->p[i];
        if (i > 0) gemm(L, pi, nrhs, c->p[i - 1], -1.0, c->Vf[i].as<double>(), 1, pi, F[i - 1].as<double>(), nrhs, 1, 1.0, F[i].as<double>(), nrhs);
        // F_i <- L_i^-1 F_i
        gemm(L, pi, nrhs, pi, 1.0, c->Li[i].as<double>(), pi, 1, F[i].as<double>(), nrhs, 1, 0.0, tmp.as<double>(), nrhs);
        CK(cudaMemcpyAsync(F[i].p, tmp.p, (size_t)pi * nrhs * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
    }
    for (int i = dm1 - 1; i >= 0; --i) {
        const int pi = c->p[i];
        if (i + 1 < dm1) {
            const int pj = c->p[i + 1];
            gemm(L, pi, nrhs, pj, -1.0, c->Vf[i + 1].as<double>(), pj, 1, F[i + 1].as<double>(), nrhs, 1, 1.0, F[i].as<double>(), nrhs);
        }
        // F_i <- L_i^-T F_i
        gemm(L, pi, nrhs, pi, 1.0, c->Li[i].as<double>(), 1, pi, F[i].as<double>(), nrhs, 1, 0.0, tmp.as<double>(), nrhs);
        CK(cudaMemcpyAsync(F[i].p, tmp.p, (size_t)pi * nrhs * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
    }
    CK(cudaStreamSynchronize(L.s));  // tmp goes back to the pool here
}

// d = 1: the pair-kernel operands straight from the tier's port matrix (port.cuh: k_single_tier_operands).
int single_tier_operands(pdn_ctx* c, Launcher& L) {
    const int m = c->m, n = c->nl;
    TierPorts& T = c->tiers[0];
    c->p0 = m;
    c->A1.alloc((size_t)m * m * sizeof(double));
    c->X0.alloc((size_t)n * m * sizeof(double));
    c->u.alloc((size_t)m * sizeof(double));
    c->w.alloc((size_t)n * sizeof(double));
    L.run(KC_DENSE, 0, [&] { k_set_identity<<<cdiv((size_t)m * m, 256), 256, 0, L.s>>>(m, c->A1.as<double>()); });
    L.run(KC_DENSE, 0, [&] { k_single_tier_operands<<<dim3(cdiv(m, 128), grid_rows((size_t)n + 1)), 128, 0, L.s>>>(m, n, T.ZT.as<double>(), T.q, T.zdiag.as<double>(), c->X0.as<double>(), c->u.as<double>(), c->w.as<double>()); });
    CK(cudaStreamSynchronize(L.s));
    return PDN_OK;
}

// S2 + S3: assemble C = [K B; B^T 0] (block-tridiagonal SPD K), factor it once, substitute for the
// m + n + (d-1) right-hand sides, eliminate the multipliers, and leave the pair-kernel operands.  The factor
// (L_i^-1, the transformed couplings, K^-1 B and S^-1) stays in the context for pdn_reff_nodes.
int recombine(pdn_ctx* c, Launcher& L) {
    if (c->d == 1) return single_tier_operands(c, L);
    const int d = c->d, dm1 = d - 1, m = c->m, n = c->nl, mn = m + n, nrhs = mn + dm1;
    std::vector<DevBuf> Kd(dm1), F(dm1), rt(dm1);
    std::vector<DevBuf>& V = c->Vf;
    std::vector<DevBuf>& Li = c->Li;
    V.clear(); V.resize(dm1);
    Li.clear(); Li.resize(dm1);
    DevBuf G, Y, fail;
    DevBuf& Sinv = c->Sinv;
    for (int i = 0; i < dm1; ++i) {
        const size_t pi = c->p[i];
        Kd[i].alloc(pi * pi * sizeof(double));
        F[i].alloc(pi * (size_t)nrhs * sizeof(double));
        if (i > 0) V[i].alloc((size_t)c->p[i - 1] * pi * sizeof(double));
        rt[i].alloc(pi * sizeof(double));
        CK(cudaMemcpyAsync(rt[i].p, c->rt[i].data(), pi * sizeof(double), cudaMemcpyHostToDevice, L.s));
    }
    G.alloc((size_t)dm1 * nrhs * sizeof(double));
    Sinv.alloc((size_t)2 * dm1 * dm1 * sizeof(double));
    Y.alloc((size_t)dm1 * mn * sizeof(double));
    fail.alloc(sizeof(int));
    CK(cudaMemsetAsync(fail.p, 0, sizeof(int), L.s));
    TierPorts& T0 = c->tiers[0];
    TierPorts& Td = c->tiers[d - 1];
    for (int i = 0; i < dm1; ++i) {
        const int pi = c->p[i];
        TierPorts& Ta = c->tiers[i];
        TierPorts& Tb = c->tiers[i + 1];
        const int oa = i > 0 ? c->p[i - 1] : 0;
        L.run(KC_DENSE, 0, [&] { k_assemble_diag<<<dim3(cdiv(pi, 128), grid_rows(pi)), 128, 0, L.s>>>(pi, Ta.ZT.as<double>(), Ta.q, oa, Tb.ZT.as<double>(), Tb.q, rt[i].as<double>(), Kd[i].as<double>()); });
        if (i + 1 < dm1) {
            const int pj = c->p[i + 1];
            L.run(KC_DENSE, 0, [&] { k_assemble_coupling<<<dim3(cdiv(pj, 128), grid_rows(pi)), 128, 0, L.s>>>(pi, pj, Tb.ZT.as<double>(), Tb.q, V[i + 1].as<double>()); });
        }
        L.run(KC_DENSE, 0, [&] { k_assemble_rhs<<<dim3(cdiv(nrhs, 128), grid_rows(pi)), 128, 0, L.s>>>(i, dm1, pi, m, n, T0.ZT.as<double>(), T0.q, T0.ntsv, Td.ZT.as<double>(), Td.q, Td.ntsv, F[i].as<double>()); });
    }
    // block-tridiagonal Cholesky.  Every diagonal factor L_i (p_i x p_i, cond ~ 1e2) is inverted once by a
    // p_i-column triangular solve; all substitutions are then K = p_i contractions on the FP64 tensor cores
    // instead of 32-wide panel solves.
    {
        DevBuf tmp;
        size_t tmax = 1;
        for (int i = 1; i < dm1; ++i) tmax = std::max(tmax, (size_t)c->p[i - 1] * c->p[i]);
        tmp.alloc(tmax * sizeof(double));
        for (int i = 0; i < dm1; ++i) {
            const int pi = c->p[i];
            if (i > 0) {
                const int ph = c->p[i - 1];
                // V_i <- L_{i-1}^-1 V_i
                gemm(L, ph, pi, ph, 1.0, Li[i - 1].as<double>(), ph, 1, V[i].as<double>(), pi, 1, 0.0, tmp.as<double>(), pi);
                CK(cudaMemcpyAsync(V[i].p, tmp.p, (size_t)ph * pi * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
                gemm(L, pi, pi, ph, -1.0, V[i].as<double>(), 1, pi, V[i].as<double>(), pi, 1, 1.0, Kd[i].as<double>(), pi);
            }
            potrf(L, Kd[i].as<double>(), pi, pi, fail.as<int>());
            Li[i].alloc((size_t)pi * pi * sizeof(double));
            L.run(KC_DENSE, 0, [&] { k_set_identity<<<cdiv((size_t)pi * pi, 256), 256, 0, L.s>>>(pi, Li[i].as<double>()); });
            trsm_fwd(L, Kd[i].as<double>(), pi, pi, Li[i].as<double>(), pi, pi);
        }
        CK(cudaStreamSynchronize(L.s));
    }
    block_substitute(c, L, F, nrhs);
    // keep K^-1 B (the last d-1 columns) for later right-hand sides
    c->KB.clear(); c->KB.resize(dm1);
    for (int i = 0; i < dm1; ++i) {
        c->KB[i].alloc((size_t)c->p[i] * dm1 * sizeof(double));
        CK(cudaMemcpy2DAsync(c->KB[i].p, (size_t)dm1 * sizeof(double), F[i].as<double>() + mn, (size_t)nrhs * sizeof(double),
                             (size_t)dm1 * sizeof(double), (size_t)c->p[i], cudaMemcpyDeviceToDevice, L.s));
    }
    // multipliers (Schur complement on the d-1 constraints, Eq. 8) and TSV currents
    for (int i = 0; i < dm1; ++i)
        L.run(KC_DENSE, 0, [&] { k_colsum<<<cdiv(nrhs, 128), 128, 0, L.s>>>(c->p[i], nrhs, F[i].as<double>(), G.as<double>() + (size_t)i * nrhs); });
    L.run(KC_DENSE, 0, [&] { k_multipliers<<<1, 256, 0, L.s>>>(dm1, mn, G.as<double>(), Sinv.as<double>(), Y.as<double>(), fail.as<int>()); });
    for (int i = 0; i < dm1; i += std::max(dm1 - 1, 1))  // only the first and the last block row are read below
        L.run(KC_DENSE, 0, [&] { k_currents<<<dim3(cdiv(mn, 128), grid_rows(c->p[i])), 128, 0, L.s>>>(c->p[i], dm1, mn, F[i].as<double>(), Y.as<double>()); });
    // operands of S4
    const int p0 = c->p[0], pd = c->p[dm1 - 1];
    c->p0 = p0;
    c->A1.alloc((size_t)m * p0 * sizeof(double));
    c->X0.alloc((size_t)n * p0 * sizeof(double));
    c->u.alloc((size_t)m * sizeof(double));
    c->w.alloc((size_t)n * sizeof(double));
    L.run(KC_DENSE, 0, [&] { k_terminal_consts<<<cdiv(m, 128), 128, 0, L.s>>>(p0, dm1, mn, m, 0, 0, T0.ZT.as<double>(), T0.q, T0.ntsv, 0, F[0].as<double>(), Y.as<double>(), T0.zdiag.as<double>(), c->u.as<double>()); });
    L.run(KC_DENSE, 0, [&] { k_terminal_consts<<<cdiv(n, 128), 128, 0, L.s>>>(pd, dm1, mn, n, m, 1, Td.ZT.as<double>(), Td.q, Td.ntsv, 0, F[dm1 - 1].as<double>(), Y.as<double>(), Td.zdiag.as<double>(), c->w.as<double>()); });
    L.run(KC_DENSE, 0, [&] { k_pack_pair_operands<<<dim3(cdiv(p0, 128), grid_rows(mn)), 128, 0, L.s>>>(p0, m, n, dm1, T0.ZT.as<double>(), T0.q, T0.ntsv, F[0].as<double>(), c->A1.as<double>(), c->X0.as<double>()); });
    if (c->terminal_pairs) {  // operands of the same-side pair kernel (port.cuh: k_pair_same)
        struct { pdn_ctx::Side& S; TierPorts& T; int p, nt, col0; double* I; } sides[2] = {
            {c->side[0], T0, p0, m, 0, F[0].as<double>()}, {c->side[1], Td, pd, n, m, F[dm1 - 1].as<double>()}};
        for (auto& sd : sides) {
            sd.S.p = sd.p;
            sd.S.A.alloc((size_t)sd.nt * sd.p * sizeof(double));
            sd.S.X.alloc((size_t)sd.nt * sd.p * sizeof(double));
            sd.S.ys.alloc((size_t)sd.nt * sizeof(double));
            sd.S.t.alloc((size_t)sd.nt * sizeof(double));
            L.run(KC_DENSE, 0, [&] { k_pack_side<<<dim3(cdiv(sd.p, 128), grid_rows(sd.nt)), 128, 0, L.s>>>(sd.p, sd.nt, sd.col0, nrhs, sd.T.ZT.as<double>(), sd.T.q, sd.T.ntsv, sd.I, sd.S.A.as<double>(), sd.S.X.as<double>()); });
            L.run(KC_DENSE, 0, [&] { k_side_consts<<<cdiv(sd.nt, 128), 128, 0, L.s>>>(sd.p, sd.nt, sd.col0, dm1, mn, sd.S.A.as<double>(), sd.S.X.as<double>(), Y.as<double>(), sd.T.zdiag.as<double>(), sd.S.ys.as<double>(), sd.S.t.as<double>()); });
        }
    }
    int h_fail = 0;
    CK(cudaMemcpyAsync(&h_fail, fail.p, sizeof(int), cudaMemcpyDeviceToHost, L.s));
    CK(cudaStreamSynchronize(L.s));
    return h_fail ? PDN_E_NUMERIC : PDN_OK;
}

}  // namespace
