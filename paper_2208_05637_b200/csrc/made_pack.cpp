// Model parameter packer — host only.  Applies the MADE masks ("MaskedFC ... removes the
// connections in the computational path of MADE") to the caller's unmasked fp32 weights; the rule is stated
// in include/nqs.h.  Device packing happens lazily in api.cu / kernels_tc.cu.
#include <new>
#include "nqs_internal.h"

extern "C" int nqs_made_create(int n_qubits, int hidden, int n_hidden_layers, const int32_t *order,
                               const int32_t *deg_hidden, const float *const *weights,
                               const float *const *biases, const float *const *phase_weights,
                               const float *const *phase_biases, nqs_made_t **out) {
    if (!out || !weights || !biases || !phase_weights || !phase_biases) return NQS_EINVAL;
    const int n = n_qubits, h = hidden, L = n_hidden_layers;
    if (n < 3 || n > NQS_MAX_QUBITS || h < 1 || h > NQS_MAX_HIDDEN || L < 1 || L > 2) return NQS_ERANGE;
    for (int k = 0; k <= L; ++k) if (!weights[k] || !biases[k]) return NQS_EINVAL;
    for (int k = 0; k < 2; ++k) if (!phase_weights[k] || !phase_biases[k]) return NQS_EINVAL;

    nqs_made *M = new (std::nothrow) nqs_made();
    if (!M) return NQS_ENOMEM;
    try {
        M->n = n; M->h = h; M->L = L; M->npad = (n + 3) & ~3;
        M->order.resize(n);
        std::vector<char> seen(n, 0);
        for (int d = 0; d < n; ++d) {
            const int q = order ? order[d] : d;
            if (q < 0 || q >= n || seen[q]) { delete M; return NQS_EINVAL; }
            seen[q] = 1; M->order[d] = q;
        }
        M->deg.resize((size_t)L * h);
        for (int k = 0; k < L; ++k)
            for (int j = 0; j < h; ++j) {
                const int d = deg_hidden ? deg_hidden[(size_t)k * h + j]
                                         : 1 + (int)(((long long)j * (n - 1)) / h);
                if (d < 1 || d > n - 1) { delete M; return NQS_ERANGE; }
                M->deg[(size_t)k * h + j] = d;
            }
        M->wm.resize(L + 1); M->bias.resize(L + 1);
        // layer 0: [h][n], M1[j][d] = deg_0[j] >= d + 1
        M->wm[0].resize((size_t)h * n);
        for (int j = 0; j < h; ++j)
            for (int d = 0; d < n; ++d)
                M->wm[0][(size_t)j * n + d] = (M->deg[j] >= d + 1) ? weights[0][(size_t)j * n + d] : 0.0f;
        M->bias[0].assign(biases[0], biases[0] + h);
        // hidden -> hidden: Mk[j'][j] = deg_k[j'] >= deg_{k-1}[j]
        for (int k = 1; k < L; ++k) {
            M->wm[k].resize((size_t)h * h);
            for (int jo = 0; jo < h; ++jo)
                for (int ji = 0; ji < h; ++ji)
                    M->wm[k][(size_t)jo * h + ji] =
                        (M->deg[(size_t)k * h + jo] >= M->deg[(size_t)(k - 1) * h + ji]) ? weights[k][(size_t)jo * h + ji] : 0.0f;
            M->bias[k].assign(biases[k], biases[k] + h);
        }
        // output: [n][h], Mout[d][j] = d + 1 > deg_{L-1}[j]
        M->wm[L].resize((size_t)n * h);
        for (int d = 0; d < n; ++d)
            for (int j = 0; j < h; ++j)
                M->wm[L][(size_t)d * h + j] = (d + 1 > M->deg[(size_t)(L - 1) * h + j]) ? weights[L][(size_t)d * h + j] : 0.0f;
        M->bias[L].assign(biases[L], biases[L] + n);
        M->p1.assign(phase_weights[0], phase_weights[0] + (size_t)h * (n - 2));
        M->p2.assign(phase_weights[1], phase_weights[1] + (size_t)4 * h);
        M->c1.assign(phase_biases[0], phase_biases[0] + h);
        M->c2.assign(phase_biases[1], phase_biases[1] + 4);
    } catch (const std::bad_alloc &) {
        delete M;
        return NQS_ENOMEM;
    }
    *out = M;
    return NQS_OK;
}

extern "C" int nqs_made_export_masked(const nqs_made_t *made, int layer, float *outp) {
    if (!made || !outp) return NQS_EINVAL;
    if (layer < 0 || layer > made->L) return NQS_ERANGE;
    const std::vector<float> &w = made->wm[layer];
    for (size_t i = 0; i < w.size(); ++i) outp[i] = w[i];
    return NQS_OK;
}
