// hadpsgd_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see hadpsgd_oracle.h).
//
// Single thread, no blocking, no fusion, no reordering: the loops below are the
// algorithm of DESIGN.md section 3 in the paper's order so a reader can check
// them against PAPER.md by eye.  Build: g++ -O2 -ffp-contract=off -fno-fast-math
// (oracle/build.py) -- -ffp-contract=off is REQUIRED so that a*b+c is two
// roundings, which is what the deterministic CUDA mode must match bit for bit.
//
// No CUDA header, no header from paper_1907_05701_b200/, nothing shared.

#include "hadpsgd_oracle.h"

#include <cstring>
#include <vector>

namespace {

// bf16 -> fp32 is exact: a bf16 value is the top 16 bits of an fp32 (R6).
inline float widen_bf16(uint16_t h) {
    uint32_t bits = static_cast<uint32_t>(h) << 16;
    float f;
    std::memcpy(&f, &bits, sizeof f);
    return f;
}

inline float load_grad(const void* grads, int grad_dtype, int64_t idx) {
    if (grad_dtype == ORACLE_GRAD_BF16) return widen_bf16(static_cast<const uint16_t*>(grads)[idx]);
    return static_cast<const float*>(grads)[idx];
}

bool build_partner(int S, uint64_t step_k, uint32_t flags, std::vector<int32_t>& partner) {
    if (S < 1) return false;
    partner.resize(S);
    if (S == 1 || (flags & ORACLE_NO_MIX)) {
        for (int s = 0; s < S; ++s) partner[s] = s;
        return true;
    }
    if (S % 2 != 0) return false;  // R8: no perfect matching => T_k of PAPER.md:66 does not exist
    if (step_k % 2 == 0) {
        for (int i = 0; i < S / 2; ++i) {  // (2i, 2i+1)
            partner[2 * i] = 2 * i + 1;
            partner[2 * i + 1] = 2 * i;
        }
    } else {
        for (int i = 0; i < S / 2; ++i) {  // (2i+1, (2i+2) mod S)
            int a = 2 * i + 1, b = (2 * i + 2) % S;
            partner[a] = b;
            partner[b] = a;
        }
    }
    return true;
}

// A caller-supplied matching (R8): an involution on {0..S-1}; partner[s] == s
// leaves s unmixed (row and column s of T_k hold a single 1).
bool copy_matching(int S, const int32_t* in, std::vector<int32_t>& partner) {
    if (S < 1 || !in) return false;
    partner.assign(in, in + S);
    for (int s = 0; s < S; ++s) {
        int p = partner[s];
        if (p < 0 || p >= S || partner[p] != s) return false;
    }
    return true;
}

void dense_T(int S, const std::vector<int32_t>& p, double* T) {
    for (int64_t k = 0; k < static_cast<int64_t>(S) * S; ++k) T[k] = 0.0;
    for (int s = 0; s < S; ++s) {
        if (p[s] == s) {
            T[static_cast<int64_t>(s) * S + s] = 1.0;
        } else {
            T[static_cast<int64_t>(s) * S + s] = 0.5;
            T[static_cast<int64_t>(s) * S + p[s]] = 0.5;
        }
    }
}

}  // namespace

extern "C" int hadpsgd_oracle_partner(int S, uint64_t step_k, int32_t* partner) {
    if (!partner) return -1;
    std::vector<int32_t> p;
    if (!build_partner(S, step_k, 0, p)) return -1;
    for (int s = 0; s < S; ++s) partner[s] = p[s];
    return 0;
}

extern "C" int hadpsgd_oracle_mixing_matrix(int S, uint64_t step_k, double* T) {
    if (!T) return -1;
    std::vector<int32_t> p;
    if (!build_partner(S, step_k, 0, p)) return -1;
    dense_T(S, p, T);
    return 0;
}

extern "C" int hadpsgd_oracle_mixing_matrix_matching(int S, const int32_t* partner, double* T) {
    if (!T) return -1;
    std::vector<int32_t> p;
    if (!copy_matching(S, partner, p)) return -1;
    dense_T(S, p, T);
    return 0;
}

namespace {

// The step for a given matching `partner` (ring or caller-supplied).
int step_f32(int S, int G, int64_t P, const void* grads, int grad_dtype, float* w, float* v,
             float lr, float mu, const std::vector<int32_t>& partner, uint32_t flags, double* diag) {
    const float invG = 1.0f / static_cast<float>(G);  // R5: mean = fp32 sum * fp32 reciprocal
    std::vector<float> u(static_cast<size_t>(S) * static_cast<size_t>(P));
    double* gsq = diag ? diag : nullptr;
    double* wsq = diag ? diag + S : nullptr;
    double* gap = diag ? diag + 2 * S : nullptr;
    if (diag)
        for (int k = 0; k < 3 * S; ++k) diag[k] = 0.0;

    // phase 1: intra-super-learner mean (eq. (6)), momentum SGD (eq. (3) + R2)
    for (int s = 0; s < S; ++s) {
        for (int64_t i = 0; i < P; ++i) {
            float acc = load_grad(grads, grad_dtype, (static_cast<int64_t>(s) * G + 0) * P + i);
            for (int g = 1; g < G; ++g)
                acc = acc + load_grad(grads, grad_dtype, (static_cast<int64_t>(s) * G + g) * P + i);
            float gbar = acc * invG;
            float t = mu * v[s * P + i];
            float vnew = t + gbar;
            v[s * P + i] = vnew;
            float t2 = lr * vnew;
            if (flags & ORACLE_EQ7_LITERAL)
                u[s * P + i] = t2;  // kept aside: subtracted AFTER mixing the old weights
            else
                u[s * P + i] = w[s * P + i] - t2;
            if (diag) gsq[s] += static_cast<double>(gbar) * static_cast<double>(gbar);
        }
    }

    // phase 2: pairwise averaging with the matched neighbour (eq. (7), T_k).
    // Diagnostics (R14): gap[s] = sum_i (a_s - a_p)^2 over the two vectors the mix
    // AVERAGES -- u_s, u_p by default; the OLD weights w_s, w_p under EQ7_LITERAL (PAPER.md:64
    // mixes Theta_k itself) -- so an unpaired member (p == s) has gap exactly 0.  wsq[s] is
    // always the sum of squares of the weights s holds AFTER the step.
    for (int s = 0; s < S; ++s) {
        int p = partner[s];
        if (p < s) continue;  // each pair once; p == s means unpaired
        for (int64_t i = 0; i < P; ++i) {
            if (flags & ORACLE_EQ7_LITERAL) {
                // Theta_{k+1} = Theta_k T_k - alpha g : mix OLD weights, subtract own update.
                // fp32 order (R14): m = 0.5f*(w_s + w_p); t = lr*v' (phase 1); w' = m - t.
                float ws = w[s * P + i], wp = w[p * P + i];
                float m = (p == s) ? ws : 0.5f * (ws + wp);
                if (diag) {
                    double d = static_cast<double>(ws) - static_cast<double>(wp);
                    gap[s] += d * d;
                }
                w[s * P + i] = m - u[s * P + i];
                if (p != s) w[p * P + i] = m - u[p * P + i];
            } else {
                float us = u[s * P + i], up = u[p * P + i];
                float m = (p == s) ? us : 0.5f * (us + up);
                if (diag) {
                    double d = static_cast<double>(us) - static_cast<double>(up);
                    gap[s] += d * d;
                }
                w[s * P + i] = m;
                if (p != s) w[p * P + i] = m;
            }
            if (diag) {
                wsq[s] += static_cast<double>(w[s * P + i]) * static_cast<double>(w[s * P + i]);
                if (p != s)
                    wsq[p] += static_cast<double>(w[p * P + i]) * static_cast<double>(w[p * P + i]);
            }
        }
        if (diag && p != s) gap[p] = gap[s];
    }
    return 0;
}

int step_f64(int S, int G, int64_t P, const void* grads, int grad_dtype, double* w, double* v,
             double lr, double mu, const std::vector<int32_t>& partner, uint32_t flags) {
    std::vector<double> u(static_cast<size_t>(S) * static_cast<size_t>(P));
    for (int s = 0; s < S; ++s) {
        for (int64_t i = 0; i < P; ++i) {
            double acc = 0.0;
            for (int g = 0; g < G; ++g)
                acc += static_cast<double>(
                    load_grad(grads, grad_dtype, (static_cast<int64_t>(s) * G + g) * P + i));
            double gbar = acc / static_cast<double>(G);
            double vnew = mu * v[s * P + i] + gbar;
            v[s * P + i] = vnew;
            if (flags & ORACLE_EQ7_LITERAL)
                u[s * P + i] = lr * vnew;
            else
                u[s * P + i] = w[s * P + i] - lr * vnew;
        }
    }
    for (int s = 0; s < S; ++s) {
        int p = partner[s];
        if (p < s) continue;
        for (int64_t i = 0; i < P; ++i) {
            if (flags & ORACLE_EQ7_LITERAL) {
                double m = (p == s) ? w[s * P + i] : 0.5 * (w[s * P + i] + w[p * P + i]);
                w[s * P + i] = m - u[s * P + i];
                if (p != s) w[p * P + i] = m - u[p * P + i];
            } else {
                double m = (p == s) ? u[s * P + i] : 0.5 * (u[s * P + i] + u[p * P + i]);
                w[s * P + i] = m;
                if (p != s) w[p * P + i] = m;
            }
        }
    }
    return 0;
}

bool args_ok(int S, int G, int64_t P, const void* grads, int grad_dtype, const void* w, const void* v) {
    if (S < 1 || G < 1 || P < 0 || !grads || !w || !v) return false;
    return grad_dtype == ORACLE_GRAD_F32 || grad_dtype == ORACLE_GRAD_BF16;
}

}  // namespace

// Ring schedule (north_star (b), R7): the matching comes from step_k's parity.
extern "C" int hadpsgd_oracle_step(int S, int G, int64_t P, const void* grads, int grad_dtype,
                                   float* w, float* v, float lr, float mu, uint64_t step_k,
                                   uint32_t flags, double* diag) {
    if (!args_ok(S, G, P, grads, grad_dtype, w, v)) return -1;
    std::vector<int32_t> partner;
    if (!build_partner(S, step_k, flags, partner)) return -1;
    return step_f32(S, G, P, grads, grad_dtype, w, v, lr, mu, partner, flags, diag);
}

extern "C" int hadpsgd_oracle_step_f64(int S, int G, int64_t P, const void* grads, int grad_dtype,
                                       double* w, double* v, double lr, double mu,
                                       uint64_t step_k, uint32_t flags) {
    if (!args_ok(S, G, P, grads, grad_dtype, w, v)) return -1;
    std::vector<int32_t> partner;
    if (!build_partner(S, step_k, flags, partner)) return -1;
    return step_f64(S, G, P, grads, grad_dtype, w, v, lr, mu, partner, flags);
}

// Caller-supplied matching (row f1, R8): any involution, unpaired members allowed (T_ss = 1).
extern "C" int hadpsgd_oracle_step_matching(int S, int G, int64_t P, const void* grads, int grad_dtype,
                                            float* w, float* v, float lr, float mu,
                                            const int32_t* partner_in, uint32_t flags, double* diag) {
    if (!args_ok(S, G, P, grads, grad_dtype, w, v)) return -1;
    std::vector<int32_t> partner;
    if (!copy_matching(S, partner_in, partner)) return -1;
    return step_f32(S, G, P, grads, grad_dtype, w, v, lr, mu, partner, flags, diag);
}

extern "C" int hadpsgd_oracle_step_matching_f64(int S, int G, int64_t P, const void* grads, int grad_dtype,
                                                double* w, double* v, double lr, double mu,
                                                const int32_t* partner_in, uint32_t flags) {
    if (!args_ok(S, G, P, grads, grad_dtype, w, v)) return -1;
    std::vector<int32_t> partner;
    if (!copy_matching(S, partner_in, partner)) return -1;
    return step_f64(S, G, P, grads, grad_dtype, w, v, lr, mu, partner, flags);
}

extern "C" int hadpsgd_oracle_round_bf16(int64_t n, const float* w, uint16_t* out) {
    if (n < 0 || !w || !out) return -1;
    for (int64_t i = 0; i < n; ++i) {
        uint32_t bits;
        std::memcpy(&bits, &w[i], sizeof bits);
        const uint32_t expo = (bits >> 23) & 0xFFu;
        if (expo == 0xFFu) {  // Inf stays Inf; NaN becomes a quiet NaN with the sign kept
            out[i] = (bits & 0x007FFFFFu) ? static_cast<uint16_t>((bits >> 16) | 0x0040u)
                                          : static_cast<uint16_t>(bits >> 16);
            continue;
        }
        // the two bf16 neighbours (same sign): magnitude truncated, and one bf16 ulp above it
        const uint32_t lo_bits = bits & 0xFFFF0000u, hi_bits = lo_bits + 0x00010000u;
        float lo, hi;
        std::memcpy(&lo, &lo_bits, sizeof lo);
        std::memcpy(&hi, &hi_bits, sizeof hi);  // may be +-Inf: overflow rounds there, as IEEE says
        // distances are exact in double (all three are fp32 values of nearby magnitude); when hi is
        // Inf the comparison uses the finite value 2^128 that Inf stands in for under IEEE rounding
        const double x = static_cast<double>(w[i]);
        const double dlo = x - static_cast<double>(lo);
        double dhi;
        if (((hi_bits >> 23) & 0xFFu) == 0xFFu) {
            const double two128 = 340282366920938463463374607431768211456.0;
            dhi = ((bits >> 31) ? -two128 : two128) - x;
        } else {
            dhi = static_cast<double>(hi) - x;
        }
        const double alo = dlo < 0 ? -dlo : dlo, ahi = dhi < 0 ? -dhi : dhi;
        uint32_t pick;
        if (alo < ahi) pick = lo_bits;
        else if (ahi < alo) pick = hi_bits;
        else pick = ((lo_bits >> 16) & 1u) ? hi_bits : lo_bits;  // tie: even last mantissa bit
        out[i] = static_cast<uint16_t>(pick >> 16);
    }
    return 0;
}

extern "C" int hadpsgd_oracle_consensus_distance(int S, int64_t P, const float* w, double* out) {
    if (S < 1 || P < 0 || !w || !out) return -1;
    double D = 0.0;
    for (int64_t i = 0; i < P; ++i) {
        double mean = 0.0;
        for (int s = 0; s < S; ++s) mean += static_cast<double>(w[s * P + i]);
        mean /= static_cast<double>(S);
        for (int s = 0; s < S; ++s) {
            double d = static_cast<double>(w[s * P + i]) - mean;
            D += d * d;
        }
    }
    *out = D;
    return 0;
}
