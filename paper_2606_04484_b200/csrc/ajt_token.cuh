// Per-token scalars of the policy loss (DESIGN.md "O-L" steps 1-6, 8 and 3b), shared by the row kernels of ajt_loss.cu and by
// the LM-head backward of ajt_lmhead.cu: one definition of the clip, the gradient gate, the KL term and the dual-clip cap.
#pragma once
#include <cuda_runtime.h>

namespace ajt {

struct TokScalars {
    float g;       // d(w L)/d logp * grad_scale
    float logp;
    float lse;
    float logS;    // log sum_v exp(z_v - M)
    float k3;      // step 8 (extended form)
    double wl;     // w * L
    double wkl;    // w * (-(logp - old))
    double wk3;    // w * k3 (extended form)
    int clip;      // bit0 high, bit1 low
};

// M = max_v z, S = sum_v exp(z_v - M) (so 1 <= S <= V), zy = z[y].  DESIGN.md O-L steps 1-6.
__device__ __forceinline__ TokScalars token_scalars(float M, float S, float zy, float old, float A, float w,
                                                    float eps_lo, float eps_hi, float grad_scale, bool use_kl = false,
                                                    float ref = 0.f, float kl_coef = 0.f, float clip_c = 0.f) {
    TokScalars o;
    const float logS = logf(S);
    o.lse = M + logS;
    o.logS = logS;
    // (zy - M) is exact for bf16 inputs; subtracting the O(1) terms first keeps the log-ratio's error ~2e-7
    const float zm = zy - M;
    o.logp = zm - logS;
    const float d = (zm - old) - logS;       // logp - old_logp
    const float r = expf(d);
    const bool hi = (A > 0.f) && (r > 1.f + eps_hi);
    const bool lo = (A < 0.f) && (r < 1.f - eps_lo);
    const float rc = fminf(fmaxf(r, 1.f - eps_lo), 1.f + eps_hi);
    float L = -fminf(r * A, rc * A);
    // step 3b (reading L-18): the dual-clip cap for negative advantages, L = min(L, -A c); no gradient where it is active
    const bool cap = clip_c > 0.f && A < 0.f && -A * clip_c < L;
    if (cap) L = -A * clip_c;
    o.g = (hi || lo || cap) ? 0.f : grad_scale * w * (-A * r);
    o.wl = (double)w * (double)L;
    o.wkl = (double)w * (-(double)d);
    o.clip = (hi ? 1 : 0) | (lo ? 2 : 0);
    o.wk3 = 0.0;
    o.k3 = 0.f;
    if (use_kl) {
        // step 8: k3 = exp(d) - d - 1, d = ref_logp - logp, clamped at 10 (low_var_kl; reading L-16)
        const float dk = (ref - zm) + logS;
        const float em1 = expm1f(dk);
        float k3 = em1 - dk;
        if (k3 < 10.f) o.g += grad_scale * w * kl_coef * (-em1);
        else k3 = 10.f;
        o.k3 = k3;
        o.wk3 = (double)w * (double)k3;
    }
    return o;
}

}  // namespace ajt
