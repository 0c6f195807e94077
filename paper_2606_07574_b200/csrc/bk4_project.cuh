// bk4_project.cuh -- the projection of one 4x4 matrix per thread, as the forward kernels call it: the lean
// iteration in warp lockstep (bk4_lean.cuh), then the guarded solver (bk4_guarded.cuh) for what that leaves, in a
// branch a warp skips when it has none.  A matrix's result depends on that matrix alone, not on which matrices
// share its warp.
#pragma once
#include "bk4_guarded.cuh"
#include "bk4_lean.cuh"


namespace bk4 {

// largest in-row logit range max_i (max_j H_ij - min_j H_ij) up to which a matrix starts from beta = 0 (above: LP
// dual start); chosen by measurement, S1.  Row offsets do not matter: eq. (10) removes them.
constexpr float kLpRange = 12.0f;
// largest in-row range up to which a narrow matrix may take the polishing step of lean_iterate (beyond, a Sinkhorn step
// is too weak to be worth the attempt: measured)
constexpr float kPolishSpread = 5.0f;

// All 32 lanes of a warp must call this together (it votes).  `valid`: this lane holds a matrix.
//   load(h)              fills h[16] with the lane's logits (called once, and again if the guarded solver is needed)
//   sm                   the lane's shared-memory scratch column (16 floats, stride kSmStride)
//   commit(out)          receives the result, original column order (NaN for a NaN/Inf matrix)
//   record(it, conv)     receives the update count and whether the tested residual reached tol_i
// GUARDED_ONLY: the lean part is skipped and every matrix takes the guarded solver.
template <bool GUARDED_ONLY, class Load, class Commit, class Record>
BK4_DEV void project_one(Load&& load, bool valid, float* sm, float tol_i, int max_iter, float lp_range, Commit&& commit,
                         Record&& record) {
    bool left = valid;  // this thread's matrix still has to be solved
    int it_lean = 0;    // updates the lean iteration spent on it
    if constexpr (!GUARDED_ONLY) {
        float h[16];
        load(h);
        // row maxima (the shift of eq. (10)) and the largest in-row range, which decides the start.
        // A NaN logit is skipped by fmaxf/fminf: such a matrix fails the first residual test and ends up in the
        // guarded solver, which reports it; an infinite logit makes the range infinite and is sent there at once.
        float rmax[4], spread = 0.0f;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            rmax[i] = fmaxf(fmaxf(h[4 * i], h[4 * i + 1]), fmaxf(h[4 * i + 2], h[4 * i + 3]));
            const float rmin = fminf(fminf(h[4 * i], h[4 * i + 1]), fminf(h[4 * i + 2], h[4 * i + 3]));
            spread = fmaxf(spread, rmax[i] - rmin);
        }
        const bool finite = valid && spread <= 3.0e38f;  // an infinite (or inf - inf = NaN) range is the guarded solver's
        bool narrow = finite && spread <= lp_range;
        float E[16], T[16], v0, v1, v2;
        bool any_narrow = __any_sync(0xffffffffu, narrow);
        if (any_narrow) {
            float s0[4];
            const float smax = narrow_exponentials(h, rmax, E, s0);
            narrow = narrow && !(smax < kPeakedSum);
            any_narrow = __any_sync(0xffffffffu, narrow);
            if (any_narrow) narrow_sweeps(E, s0, v0, v1, v2);
        }
        const bool wide = finite && !narrow, active = finite;
        const bool any_wide = __any_sync(0xffffffffu, wide);
        const bool polishable = narrow && spread <= kPolishSpread;  // see lean_iterate
        if (any_narrow || any_wide) {
            LeanResult res;
            if (any_wide) {
                // the wide start works on column-permuted matrices: a narrow matrix in the same warp keeps its order
                unsigned code;
                if (!any_narrow) {
                    wide_start(h, sm, E, v0, v1, v2, code);  // straight into E: a warp of wide matrices moves no registers
                } else {
                    float Ew[16], w0, w1, w2;
                    wide_start(h, sm, Ew, w0, w1, w2, code);
                    if (wide) {
#pragma unroll
                        for (int q = 0; q < 16; ++q) E[q] = Ew[q];
                        v0 = w0, v1 = w1, v2 = w2;
                    } else {
                        code = kIdentityCode;
                    }
                }
                const bool plain3 = wide && max_iter >= kLeanFreeWide;
                res = any_narrow ? lean_iterate<kLeanMixed>(E, v0, v1, v2, active, plain3, polishable, tol_i, max_iter, T)
                                 : lean_iterate<kLeanWide>(E, v0, v1, v2, active, plain3, false, tol_i, max_iter, T);
                if (active && res.stored) {
                    float out[16];
                    clamp_diagonal(T);
                    unpermute_columns(T, code, sm, out);
                    commit(out);
                }
            } else {
                res = lean_iterate<kLeanNarrow>(E, v0, v1, v2, active, false, polishable, tol_i, max_iter, T);
                if (active && res.stored) {
                    clamp_diagonal(T);
                    commit(T);
                }
            }
            if (active && res.stored) record(res.it, res.converged);
            left = valid && !(active && res.stored);
            it_lean = active ? res.it : 0;
        }
    }
    if (__any_sync(0xffffffffu, left)) {
        if (left) {  // every lane for itself: this is the rare path
            float h[16];
            load(h);  // the lean part has stored only matrices this branch does not touch
            float poison = 0.0f;
#pragma unroll
            for (int q = 0; q < 16; ++q) poison = __fmaf_rn(h[q], 0.0f, poison);  // NaN iff some logit is NaN or +-Inf
            const bool bad = !(poison == 0.0f);
            // LP dual potentials and the column permutation (a NaN/Inf matrix goes through the motions and is
            // overwritten with NaN)
            float w[4][4], xs[4], hc[16];
            unsigned code;
            lp_dual(h, sm, w, xs, code);
            gather_columns(sm, code, hc);
            auto gather = [&](float(&Hr)[16]) {
                float hr[16];
                load(hr);
#pragma unroll
                for (int q = 0; q < 16; ++q) sm[q * kSmStride] = hr[q];
                gather_columns(sm, code, Hr);
            };
            auto emit = [&](const float(&T)[16], int iters, bool converged) {
                float Tc[16], out[16];
#pragma unroll
                for (int q = 0; q < 16; ++q) Tc[q] = T[q];
                clamp_diagonal(Tc);
                unpermute_columns(Tc, code, sm, out);
#pragma unroll
                for (int q = 0; q < 16; ++q) out[q] = bad ? kNaN : out[q];
                commit(out);
                record(it_lean + iters, converged && !bad);
            };
            newton_guarded(hc, xs, tol_i, max_iter > it_lean ? max_iter - it_lean : 0, gather, emit);
        }
    }
}

}  // namespace bk4
