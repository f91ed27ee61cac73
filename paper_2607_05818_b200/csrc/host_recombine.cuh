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
// S2 + S3: assemble C = [K B; B^T 0] (block-tridiagonal SPD K), factor it once, substitute for the
// m + n + (d-1) right-hand sides, eliminate the multipliers, and leave the pair-kernel operands.
int recombine(pdn_ctx* c, Launcher& L) {
    const int d = c->d, dm1 = d - 1, m = c->m, n = c->nl, mn = m + n, nrhs = mn + dm1;
    std::vector<DevBuf> Kd(dm1), V(dm1), F(dm1), rt(dm1);
    DevBuf G, Sinv, Y, fail;
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
        L.run(KC_DENSE, 0, [&] { k_assemble_diag<<<dim3(cdiv(pi, 128), pi), 128, 0, L.s>>>(pi, Ta.ZT.as<double>(), Ta.q, oa, Tb.ZT.as<double>(), Tb.q, rt[i].as<double>(), Kd[i].as<double>()); });
        if (i + 1 < dm1) {
            const int pj = c->p[i + 1];
            L.run(KC_DENSE, 0, [&] { k_assemble_coupling<<<dim3(cdiv(pj, 128), pi), 128, 0, L.s>>>(pi, pj, Tb.ZT.as<double>(), Tb.q, V[i + 1].as<double>()); });
        }
        L.run(KC_DENSE, 0, [&] { k_assemble_rhs<<<dim3(cdiv(nrhs, 128), pi), 128, 0, L.s>>>(i, dm1, pi, m, n, T0.ZT.as<double>(), T0.q, T0.ntsv, Td.ZT.as<double>(), Td.q, Td.ntsv, F[i].as<double>()); });
    }
    // block-tridiagonal Cholesky + forward substitution.  Every diagonal factor L_i (p_i x p_i, cond ~ 1e2) is
    // inverted once by a p_i-column triangular solve; all substitutions for the m + n + d-1 right-hand sides
    // are then K = p_i contractions on the FP64 tensor cores instead of 32-wide panel solves.
    std::vector<DevBuf> Li(dm1);
    DevBuf tmp;
    {
        size_t tmax = 0;
        for (int i = 0; i < dm1; ++i) tmax = std::max(tmax, (size_t)c->p[i] * std::max(nrhs, c->p[i]));
        for (int i = 1; i < dm1; ++i) tmax = std::max(tmax, (size_t)c->p[i - 1] * c->p[i]);
        tmp.alloc(tmax * sizeof(double));
    }
    for (int i = 0; i < dm1; ++i) {
        const int pi = c->p[i];
        if (i > 0) {
            const int ph = c->p[i - 1];
            // V_i <- L_{i-1}^-1 V_i
            gemm(L, ph, pi, ph, 1.0, Li[i - 1].as<double>(), ph, 1, V[i].as<double>(), pi, 1, 0.0, tmp.as<double>(), pi);
            CK(cudaMemcpyAsync(V[i].p, tmp.p, (size_t)ph * pi * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
            gemm(L, pi, pi, ph, -1.0, V[i].as<double>(), 1, pi, V[i].as<double>(), pi, 1, 1.0, Kd[i].as<double>(), pi);
            gemm(L, pi, nrhs, ph, -1.0, V[i].as<double>(), 1, pi, F[i - 1].as<double>(), nrhs, 1, 1.0, F[i].as<double>(), nrhs);
        }
        potrf(L, Kd[i].as<double>(), pi, pi, fail.as<int>());
        Li[i].alloc((size_t)pi * pi * sizeof(double));
        L.run(KC_DENSE, 0, [&] { k_set_identity<<<cdiv((size_t)pi * pi, 256), 256, 0, L.s>>>(pi, Li[i].as<double>()); });
        trsm_fwd(L, Kd[i].as<double>(), pi, pi, Li[i].as<double>(), pi, pi);
        // F_i <- L_i^-1 F_i
        gemm(L, pi, nrhs, pi, 1.0, Li[i].as<double>(), pi, 1, F[i].as<double>(), nrhs, 1, 0.0, tmp.as<double>(), nrhs);
        CK(cudaMemcpyAsync(F[i].p, tmp.p, (size_t)pi * nrhs * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
    }
    // backward substitution
    for (int i = dm1 - 1; i >= 0; --i) {
        const int pi = c->p[i];
        if (i + 1 < dm1) {
            const int pj = c->p[i + 1];
            gemm(L, pi, nrhs, pj, -1.0, V[i + 1].as<double>(), pj, 1, F[i + 1].as<double>(), nrhs, 1, 1.0, F[i].as<double>(), nrhs);
        }
        // F_i <- L_i^-T F_i
        gemm(L, pi, nrhs, pi, 1.0, Li[i].as<double>(), 1, pi, F[i].as<double>(), nrhs, 1, 0.0, tmp.as<double>(), nrhs);
        CK(cudaMemcpyAsync(F[i].p, tmp.p, (size_t)pi * nrhs * sizeof(double), cudaMemcpyDeviceToDevice, L.s));
    }
    // multipliers (Schur complement on the d-1 constraints, Eq. 8) and TSV currents
    for (int i = 0; i < dm1; ++i)
        L.run(KC_DENSE, 0, [&] { k_colsum<<<cdiv(nrhs, 128), 128, 0, L.s>>>(c->p[i], nrhs, F[i].as<double>(), G.as<double>() + (size_t)i * nrhs); });
    L.run(KC_DENSE, 0, [&] { k_multipliers<<<1, 256, 0, L.s>>>(dm1, mn, G.as<double>(), Sinv.as<double>(), Y.as<double>(), fail.as<int>()); });
    for (int i = 0; i < dm1; i += std::max(dm1 - 1, 1))  // only the first and the last block row are read below
        L.run(KC_DENSE, 0, [&] { k_currents<<<dim3(cdiv(mn, 128), c->p[i]), 128, 0, L.s>>>(c->p[i], dm1, mn, F[i].as<double>(), Y.as<double>()); });
    // operands of S4
    const int p0 = c->p[0], pd = c->p[dm1 - 1];
    c->p0 = p0;
    c->A1.alloc((size_t)m * p0 * sizeof(double));
    c->X0.alloc((size_t)n * p0 * sizeof(double));
    c->u.alloc((size_t)m * sizeof(double));
    c->w.alloc((size_t)n * sizeof(double));
    L.run(KC_DENSE, 0, [&] { k_terminal_consts<<<cdiv(m, 128), 128, 0, L.s>>>(p0, dm1, mn, m, 0, 0, T0.ZT.as<double>(), T0.q, T0.ntsv, 0, F[0].as<double>(), Y.as<double>(), T0.zdiag.as<double>(), c->u.as<double>()); });
    L.run(KC_DENSE, 0, [&] { k_terminal_consts<<<cdiv(n, 128), 128, 0, L.s>>>(pd, dm1, mn, n, m, 1, Td.ZT.as<double>(), Td.q, Td.ntsv, 0, F[dm1 - 1].as<double>(), Y.as<double>(), Td.zdiag.as<double>(), c->w.as<double>()); });
    L.run(KC_DENSE, 0, [&] { k_pack_pair_operands<<<dim3(cdiv(p0, 128), mn), 128, 0, L.s>>>(p0, m, n, dm1, T0.ZT.as<double>(), T0.q, T0.ntsv, F[0].as<double>(), c->A1.as<double>(), c->X0.as<double>()); });
    if (c->terminal_pairs) {  // operands of the same-side pair kernel (port.cuh: k_pair_same)
        struct { pdn_ctx::Side& S; TierPorts& T; int p, nt, col0; double* I; } sides[2] = {
            {c->side[0], T0, p0, m, 0, F[0].as<double>()}, {c->side[1], Td, pd, n, m, F[dm1 - 1].as<double>()}};
        for (auto& sd : sides) {
            sd.S.p = sd.p;
            sd.S.A.alloc((size_t)sd.nt * sd.p * sizeof(double));
            sd.S.X.alloc((size_t)sd.nt * sd.p * sizeof(double));
            sd.S.ys.alloc((size_t)sd.nt * sizeof(double));
            sd.S.t.alloc((size_t)sd.nt * sizeof(double));
            L.run(KC_DENSE, 0, [&] { k_pack_side<<<dim3(cdiv(sd.p, 128), sd.nt), 128, 0, L.s>>>(sd.p, sd.nt, sd.col0, nrhs, sd.T.ZT.as<double>(), sd.T.q, sd.T.ntsv, sd.I, sd.S.A.as<double>(), sd.S.X.as<double>()); });
            L.run(KC_DENSE, 0, [&] { k_side_consts<<<cdiv(sd.nt, 128), 128, 0, L.s>>>(sd.p, sd.nt, sd.col0, dm1, mn, sd.S.A.as<double>(), sd.S.X.as<double>(), Y.as<double>(), sd.T.zdiag.as<double>(), sd.S.ys.as<double>(), sd.S.t.as<double>()); });
        }
    }
    int h_fail = 0;
    CK(cudaMemcpyAsync(&h_fail, fail.p, sizeof(int), cudaMemcpyDeviceToHost, L.s));
    CK(cudaStreamSynchronize(L.s));
    return h_fail ? PDN_E_NUMERIC : PDN_OK;
}

}  // namespace
