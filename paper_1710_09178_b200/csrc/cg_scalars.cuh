// cg_scalars.cuh -- the scalar recurrences of the multishift CG, evaluated on the
// device by the last block of the reduction that produces their input, so that an iteration never
// returns to the host.  Thread k handles shift k (blockDim >= kMaxShifts).
#pragma once
#include "internal.cuh"

namespace qcd {

// After pAp = Re<p_0, q> is known:
//   alpha = rho / pAp
//   zeta_k^new = zeta_k zeta_k^old alpha_old / ( alpha beta_old (zeta_k^old - zeta_k)
//                                               + zeta_k^old alpha_old (1 + delta_k alpha) )
//   alpha_k = alpha zeta_k^new / zeta_k
__device__ __forceinline__ void cg_step_alpha(CgState *st, double pAp)
{
    const int k = threadIdx.x;
    const double alpha = st->rho / pAp;
    if (k < st->nshift && st->active[k]) {
        const double delta = st->sigma[k] - st->sigma[0];
        const double z = st->zeta[k], zo = st->zeta_old[k];
        const double ao = st->alpha_old, bo = st->beta_old;
        const double zn = z * zo * ao / (alpha * bo * (zo - z) + zo * ao * (1.0 + delta * alpha));
        st->zeta_new[k] = zn;
        st->coef_a[k] = alpha * zn / z;
    }
    if (k == 0) {
        st->pAp = pAp;
        st->alpha = alpha;
    }
}

// After rho' = <r,r> of the updated residual is known:
//   beta = rho'/rho ; beta_k = beta (zeta_k^new/zeta_k)^2 ; p_k = zeta_k^new r + beta_k p_k
//   rotate zeta ; freeze k > 0 when |zeta_k| sqrt(rho') <= f tol sqrt(rho_b) ; stop test (C10, C13)
__device__ __forceinline__ void cg_step_beta(CgState *st, double rho_new)
{
    __shared__ int s_act[kMaxShifts];
    const int k = threadIdx.x;
    const int n = st->nshift;
    const double rho = st->rho, rho_b = st->rho_b;
    const double beta = rho_new / rho;
    const int slot = st->iter % st->defer;       // this is iteration st->iter + 1: slot (n - 1) % defer
    if (k < n) {
        const int a = st->active[k];
        s_act[k] = a;
        st->hist_on[slot][k] = a;
        if (a) {
            const double z = st->zeta[k], zn = st->zeta_new[k];
            const double ratio = zn / z;
            st->coef_z[k] = zn;
            st->coef_b[k] = beta * ratio * ratio;
            st->hist_a[slot][k] = st->coef_a[k];     // written by this thread in cg_step_alpha
            st->hist_z[slot][k] = zn;
            st->hist_b[slot][k] = beta * ratio * ratio;
            st->zeta_old[k] = z;
            st->zeta[k] = zn;
            if (k > 0 && fabs(zn) * sqrt(rho_new) <= st->freeze * st->tol * sqrt(rho_b))
                st->active[k] = 0;
        }
    }
    __syncthreads();
    if (k == 0) {
        int m = 0;
        for (int j = 0; j < n; ++j)
            if (s_act[j]) st->list[m++] = j;   // shifts the update kernel touches this iteration
        st->nlist = m;
        st->alpha_old = st->alpha;
        st->beta_old = beta;
        st->beta = beta;
        st->rho = rho_new;
        const int it = st->iter + 1;
        st->iter = it;
        if (sqrt(rho_new / rho_b) <= st->tol || it >= st->max_iter) st->done = 1;
    }
}

}  // namespace qcd
