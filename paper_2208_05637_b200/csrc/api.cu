// C-ABI glue: device upload, workspace, mini-batch scheduler (a7), statistics (a6), error strings.
#include <cstring>
#include <new>
#include "nqs_internal.h"

long long g_launch_count = 0;

#define CU(x) do { if ((x) != cudaSuccess) return NQS_ECUDA; } while (0)

int nqs_check_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
    return major == 10 ? NQS_OK : NQS_EARCH;
}

template <class T>
static int upload(const T *src, size_t count, void **dst) {
    *dst = nullptr;
    if (cudaMalloc(dst, sizeof(T) * (count ? count : 1)) != cudaSuccess) { cudaGetLastError(); return NQS_ENOMEM; }
    if (count && cudaMemcpy(*dst, src, sizeof(T) * count, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError(); cudaFree(*dst); *dst = nullptr;
        return NQS_ECUDA;
    }
    return NQS_OK;
}

static int same_device(int recorded) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
    return dev == recorded ? NQS_OK : NQS_EINVAL;
}

int nqs_ham_upload(const nqs_ham *H) {
    if (H->on_device) return same_device(H->device);
    int rc = nqs_check_device();
    if (rc) return rc;
    cudaGetDevice(&H->device);
    // c_t * (-i)^{r_t}  (Eq. 16 prefactor folded into the coefficient)
    std::vector<float2> cph((size_t)H->K);
    for (int64_t t = 0; t < H->K; ++t) {
        const float c = H->coef[t];
        switch (H->ycount[t] & 3) {
            case 0: cph[t] = make_float2(c, 0.f); break;
            case 1: cph[t] = make_float2(0.f, -c); break;
            case 2: cph[t] = make_float2(-c, 0.f); break;
            default: cph[t] = make_float2(0.f, c); break;
        }
    }
    if ((rc = upload(H->flips.data(), H->flips.size(), &H->d_flips)) == NQS_OK &&
        (rc = upload(H->offsets.data(), H->offsets.size(), &H->d_offsets)) == NQS_OK &&
        (rc = upload(H->zy.data(), H->zy.size(), &H->d_zy)) == NQS_OK &&
        (rc = upload(cph.data(), cph.size(), &H->d_cph)) == NQS_OK) {
        H->on_device = true;
        return NQS_OK;
    }
    // a partial upload is released: the handle stays usable for a later attempt
    if (H->d_flips) cudaFree(H->d_flips);
    if (H->d_offsets) cudaFree(H->d_offsets);
    if (H->d_zy) cudaFree(H->d_zy);
    if (H->d_cph) cudaFree(H->d_cph);
    H->d_flips = H->d_offsets = H->d_zy = H->d_cph = nullptr;
    return rc;
}

HamDev nqs_ham_dev(const nqs_ham *H) {
    HamDev d;
    d.n = H->n; d.K = H->K; d.G = H->G;
    d.flips = (const ulonglong2 *)H->d_flips; d.offsets = (const uint32_t *)H->d_offsets;
    d.zy = (const ulonglong2 *)H->d_zy; d.cph = (const float2 *)H->d_cph;
    d.has_diag = (H->G > 0 && H->flips[0] == 0 && H->flips[1] == 0) ? 1 : 0;
    return d;
}

extern "C" void nqs_ham_free(nqs_ham_t *H) {
    if (!H) return;
    if (H->on_device) { cudaFree(H->d_flips); cudaFree(H->d_offsets); cudaFree(H->d_zy); cudaFree(H->d_cph); }
    delete H;
}

static int made_upload_tensors(const nqs_made *M);

int nqs_made_upload(const nqs_made *M) {
    if (M->on_device) return same_device(M->device);
    int rc = nqs_check_device();
    if (rc) return rc;
    cudaGetDevice(&M->device);
    if ((rc = made_upload_tensors(M))) {
        // a partial upload is released: the handle stays usable for a later attempt and holds nothing twice
        for (void *p : M->d_allocs) cudaFree(p);
        M->d_allocs.clear();
        M->dev = MadeDev{};
        return rc;
    }
    // The tensor-core pack is optional: if it cannot be built or uploaded the handle still serves NQS_PATH_SIMT,
    // NQS_PATH_AUTO takes that path and a forced NQS_PATH_TC reports NQS_EUNSUPPORTED (include/nqs.h).
    if (tc_supported(M) && tc_pack_upload(M) != NQS_OK) { cudaGetLastError(); M->tc_failed = true; }
    M->on_device = true;
    return NQS_OK;
}

static int made_upload_tensors(const nqs_made *M) {
    int rc = NQS_OK;
    const int n = M->n, h = M->h, L = M->L, npad = M->npad;
    auto up = [&](const std::vector<float> &v, const float **dst) -> int {
        void *p = nullptr;
        int r = upload(v.data(), v.size(), &p);
        if (r) return r;
        M->d_allocs.push_back(p);
        *dst = (const float *)p;
        return NQS_OK;
    };
    MadeDev &d = M->dev;
    d.n = n; d.h = h; d.L = L; d.npad = npad;
    d.n_up = M->n_up; d.n_down = M->n_down;
    d.spin_lo = d.spin_hi = 0;
    for (int k = 0; k < n; ++k)
        if (M->order[k] & 1) { if (k < 64) d.spin_lo |= 1ull << k; else d.spin_hi |= 1ull << (k - 64); }
    {
        void *p = nullptr;
        if ((rc = upload(M->order.data(), M->order.size(), &p))) return rc;
        M->d_allocs.push_back(p); d.order = (const int32_t *)p;
    }
    std::vector<float> t;
    t.assign((size_t)n * h, 0.f);                                      // w1t [n][h]
    for (int j = 0; j < h; ++j) for (int k = 0; k < n; ++k) t[(size_t)k * h + j] = M->wm[0][(size_t)j * n + k];
    if ((rc = up(t, &d.w1t))) return rc;
    d.w2t = nullptr; d.b2 = nullptr;
    if (L == 2) {
        t.assign((size_t)h * h, 0.f);                                  // w2t [h][h]
        for (int j = 0; j < h; ++j) for (int k = 0; k < h; ++k) t[(size_t)k * h + j] = M->wm[1][(size_t)j * h + k];
        if ((rc = up(t, &d.w2t))) return rc;
        if ((rc = up(M->bias[1], &d.b2))) return rc;
    }
    t.assign((size_t)h * npad, 0.f);                                   // w3t [h][npad]
    for (int dd = 0; dd < n; ++dd) for (int k = 0; k < h; ++k) t[(size_t)k * npad + dd] = M->wm[L][(size_t)dd * h + k];
    if ((rc = up(t, &d.w3t))) return rc;
    if ((rc = up(M->bias[0], &d.b1))) return rc;
    t.assign(npad, 0.f);
    for (int dd = 0; dd < n; ++dd) t[dd] = M->bias[L][dd];
    if ((rc = up(t, &d.b3))) return rc;
    t.assign((size_t)n * h, 0.f);                                      // p1t [n][h], last two input rows zero
    for (int j = 0; j < h; ++j) for (int k = 0; k < n - 2; ++k) t[(size_t)k * h + j] = M->p1[(size_t)j * (n - 2) + k];
    if ((rc = up(t, &d.p1t))) return rc;
    t.assign((size_t)h * 4, 0.f);                                      // p2t [h][4]
    for (int o = 0; o < 4; ++o) for (int k = 0; k < h; ++k) t[(size_t)k * 4 + o] = M->p2[(size_t)o * h + k];
    if ((rc = up(t, &d.p2t))) return rc;
    if ((rc = up(M->c1, &d.c1))) return rc;
    if ((rc = up(M->c2, &d.c2))) return rc;
    {   // kend arrays (see MadeDev)
        auto kend_of = [&](const std::vector<float> &W, int rows, int cols, const int32_t **dst) -> int {
            std::vector<int32_t> ke((size_t)rows, 0);
            for (int j = 0; j < rows; ++j)
                for (int k = cols - 1; k >= 0; --k)
                    if (W[(size_t)j * cols + k] != 0.0f) { ke[j] = k + 1; break; }
            void *p = nullptr;
            const int r = upload(ke.data(), ke.size(), &p);
            if (r) return r;
            M->d_allocs.push_back(p);
            *dst = (const int32_t *)p;
            return NQS_OK;
        };
        d.kend2 = nullptr;
        if ((rc = kend_of(M->wm[0], h, n, &d.kend1))) return rc;
        if (L == 2 && (rc = kend_of(M->wm[1], h, h, &d.kend2))) return rc;
        if ((rc = kend_of(M->wm[L], n, h, &d.kend3))) return rc;
    }
    return NQS_OK;
}

int nqs_ws_reserve(const nqs_made *M, size_t bytes) {
    if (M->ws_bytes >= bytes) return NQS_OK;
    if (M->ws) { cudaFree(M->ws); M->ws = nullptr; M->ws_bytes = 0; }
    if (cudaMalloc(&M->ws, bytes) != cudaSuccess) { cudaGetLastError(); return NQS_ENOMEM; }
    M->ws_bytes = bytes;
    return NQS_OK;
}

extern "C" int nqs_made_set_constraint(nqs_made_t *M, int n_up, int n_down) {
    if (!M) return NQS_EINVAL;
    if ((n_up < 0) != (n_down < 0)) return NQS_EINVAL;
    if (n_up < 0) { n_up = n_down = -1; }
    else if (n_up > (M->n + 1) / 2 || n_down > M->n / 2) return NQS_EINVAL;       // even qubits = up, odd = down (Eq. 12)
    M->n_up = n_up; M->n_down = n_down;
    M->dev.n_up = n_up; M->dev.n_down = n_down;                                   // the device view is passed by value per launch
    return NQS_OK;
}

extern "C" void nqs_made_free(nqs_made_t *M) {
    if (!M) return;
    for (void *p : M->d_allocs) cudaFree(p);
    if (M->ws) cudaFree(M->ws);
    if (M->hx) cudaFree(M->hx);
    if (M->hc) cudaFree(M->hc);
    if (M->he) cudaFree(M->he);
    if (M->samp_ws) cudaFree(M->samp_ws);
    if (M->h_stream) cudaStreamDestroy(M->h_stream);
    for (cudaEvent_t e : M->ev) cudaEventDestroy(e);
    tc_pack_free(M);
    grad_pack_free(M);
    delete M;
}

// The shape decides, except that a handle whose tensor-core pack failed to upload (tc_failed, known once
// nqs_made_upload has run) is an fp32-path handle: callers resolve again after the upload.
static int resolve_path(const nqs_made *M, int path, int *use_tc) {
    const bool tc_ok = tc_supported(M) && !M->tc_failed;
    if (path == NQS_PATH_SIMT) { *use_tc = 0; return NQS_OK; }
    if (path == NQS_PATH_TC) { if (!tc_ok) return NQS_EUNSUPPORTED; *use_tc = 1; return NQS_OK; }
    if (path == NQS_PATH_AUTO) { *use_tc = tc_ok ? 1 : 0; return NQS_OK; }
    return NQS_EINVAL;
}

extern "C" int nqs_made_path(const nqs_made_t *M, int path) {
    if (!M) return NQS_EINVAL;
    int use_tc = 0;
    const int rc = resolve_path(M, path, &use_tc);
    return rc ? rc : (use_tc ? NQS_PATH_TC : NQS_PATH_SIMT);
}

extern "C" int nqs_made_tc_flops(const nqs_made_t *M, int64_t *issued_per_eval, int64_t *dense_per_eval) {
    if (!M || !issued_per_eval || !dense_per_eval) return NQS_EINVAL;
    if (!tc_supported(M)) return NQS_EUNSUPPORTED;
    const int rc = nqs_made_upload(M);
    if (rc) return rc;
    if (!M->tc) return NQS_EUNSUPPORTED;
    long long issued = 0, dense = 0;
    tc_mma_counts(M, &issued, &dense);             // in units of one K-step (16) x one output column, per row
    *issued_per_eval = 32 * issued;
    *dense_per_eval = 32 * dense;
    return NQS_OK;
}

extern "C" int nqs_made_logpsi(const nqs_made_t *M, const uint64_t *configs_dev, int64_t B, float *out_dev,
                               int path, void *cuda_stream) {
    if (!M || B < 0 || (B > 0 && (!configs_dev || !out_dev))) return NQS_EINVAL;
    int use_tc = 0;
    int rc = resolve_path(M, path, &use_tc);
    if (rc) return rc;
    if (B == 0) return NQS_OK;
    if ((rc = nqs_made_upload(M))) return rc;
    if ((rc = resolve_path(M, path, &use_tc))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (use_tc) return launch_logpsi_tc(M, (const ulonglong2 *)configs_dev, B, (float2 *)out_dev, st);
    return launch_logpsi_simt(M->dev, (const ulonglong2 *)configs_dev, B, (float2 *)out_dev, st);
}

extern "C" int nqs_pauli_contract(const nqs_ham_t *H, const uint64_t *samples_dev, int64_t B, int64_t g0,
                                  int64_t g1, float *S_out_dev, void *cuda_stream) {
    if (!H || B < 0 || g0 < 0 || g1 < g0 || g1 > H->G) return NQS_EINVAL;
    if (B == 0 || g1 == g0) return NQS_OK;
    if (!samples_dev || !S_out_dev) return NQS_EINVAL;
    int rc = nqs_ham_upload(H);
    if (rc) return rc;
    return launch_contract(nqs_ham_dev(H), (const ulonglong2 *)samples_dev, B, g0, g1, (float2 *)S_out_dev,
                           (cudaStream_t)cuda_stream);
}

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

extern "C" int nqs_local_energy(const nqs_ham_t *H, const nqs_made_t *M, const uint64_t *samples_dev,
                                const int64_t *counts_dev, int64_t B, int64_t minibatch, int path,
                                float *eloc_out_dev, double *stats_out_host, void *cuda_stream) {
    if (!H || !M || B < 0 || minibatch < 0) return NQS_EINVAL;
    if (H->n != M->n) return NQS_EINVAL;
    int use_tc = 0;
    int rc = resolve_path(M, path, &use_tc);
    if (rc) return rc;
    if (B == 0) {
        if (stats_out_host) for (int k = 0; k < 5; ++k) stats_out_host[k] = 0.0;
        return NQS_OK;
    }
    if (!samples_dev || !eloc_out_dev) return NQS_EINVAL;
    if ((rc = nqs_ham_upload(H))) return rc;
    if ((rc = nqs_made_upload(M))) return rc;
    if ((rc = resolve_path(M, path, &use_tc))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const HamDev hm = nqs_ham_dev(H);
    const long long mb = minibatch > 0 ? minibatch : 8192;
    const long long mb_eff = mb < B ? mb : B;
    const int n_mb = (int)((B + mb - 1) / mb);

    // workspace: [stats 4 doubles | max-ratio bits | base logpsi | per-path scratch]
    int nsplit = 1;
    const size_t scratch = use_tc ? eloc_tc_ws_bytes(mb_eff, hm) : eloc_simt_partial_bytes(mb_eff, &nsplit, hm);
    const size_t off_base = 256, off_scratch = off_base + align256(sizeof(float2) * (size_t)mb_eff);
    if ((rc = nqs_ws_reserve(M, off_scratch + align256(scratch)))) return rc;
    unsigned char *ws = (unsigned char *)M->ws;
    double *d_stats = (double *)ws;
    unsigned *d_maxr = (unsigned *)(ws + 64);
    float2 *d_base = (float2 *)(ws + off_base);
    void *d_scratch = ws + off_scratch;
    CU(cudaMemsetAsync(ws, 0, 128, st));

    while ((int)M->ev.size() < 2 * n_mb) {
        cudaEvent_t e;
        CU(cudaEventCreate(&e));
        M->ev.push_back(e);
    }
    M->ev_used = 0;

    for (int b = 0; b < n_mb; ++b) {                                    // (a7) PAPER.md:202
        const long long i0 = (long long)b * mb, nb = (B - i0 < mb) ? (B - i0) : mb;
        const ulonglong2 *xs = (const ulonglong2 *)samples_dev + i0;
        float2 *eo = (float2 *)eloc_out_dev + i0;
        // base amplitudes f(x) (Alg. 1 line 2), same arithmetic path as the connected ones
        if (use_tc) rc = launch_logpsi_tc(M, xs, nb, d_base, st);
        else        rc = launch_logpsi_simt(M->dev, xs, nb, d_base, st);
        if (rc) return rc;
        CU(cudaEventRecord(M->ev[2 * b], st));
        if (use_tc) rc = launch_eloc_tc(hm, M, xs, d_base, nb, eo, d_maxr, st);
        else        rc = launch_eloc_simt(hm, M->dev, xs, d_base, nb, eo, (float2 *)d_scratch, nsplit, d_maxr, st);
        if (rc) return rc;
        CU(cudaEventRecord(M->ev[2 * b + 1], st));
        M->ev_used = b + 1;
        if (stats_out_host) {
            if ((rc = launch_stats(eo, counts_dev ? (const long long *)counts_dev + i0 : nullptr, nb, d_stats, st))) return rc;
        }
    }
    if (stats_out_host) {
        double s4[4]; unsigned mr = 0;
        CU(cudaMemcpyAsync(s4, d_stats, sizeof(s4), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(&mr, d_maxr, sizeof(mr), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        float mrf; memcpy(&mrf, &mr, 4);
        for (int k = 0; k < 4; ++k) stats_out_host[k] = s4[k];
        stats_out_host[4] = (double)mrf;
    }
    return NQS_OK;
}

extern "C" int nqs_local_energy_host(const nqs_ham_t *H, const nqs_made_t *M, const uint64_t *samples_host,
                                     const int64_t *counts_host, int64_t B, int64_t minibatch, int path,
                                     float *eloc_out_host, double *stats_out_host) {
    if (!H || !M || B < 0) return NQS_EINVAL;
    if (B == 0) return nqs_local_energy(H, M, nullptr, nullptr, 0, minibatch, path, nullptr, stats_out_host, nullptr);
    if (!samples_host || !eloc_out_host) return NQS_EINVAL;
    {   // bits >= n_qubits must be zero (include/nqs.h): checked here, where the samples are host memory
        const int n = M->n;
        const uint64_t lo_bad = n >= 64 ? 0ull : ~0ull << n, hi_bad = n >= 128 ? 0ull : (n <= 64 ? ~0ull : ~0ull << (n - 64));
        for (int64_t i = 0; i < B; ++i)
            if ((samples_host[2 * i] & lo_bad) | (samples_host[2 * i + 1] & hi_bad)) return NQS_EINVAL;
        if (H->n != n) return NQS_EINVAL;
    }
    int rc = nqs_check_device();
    if (rc) return rc;
    // staging buffers and the stream live in the model handle and are reused (a handle serves one call at a time)
    if (!M->h_stream && cudaStreamCreateWithFlags(&M->h_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
    if (M->h_rows < (size_t)B) {
        if (M->hx) cudaFree(M->hx);
        if (M->hc) cudaFree(M->hc);
        if (M->he) cudaFree(M->he);
        M->hx = M->hc = M->he = nullptr; M->h_rows = 0;
        if (cudaMalloc(&M->hx, 16 * (size_t)B) != cudaSuccess || cudaMalloc(&M->he, 8 * (size_t)B) != cudaSuccess ||
            cudaMalloc(&M->hc, 8 * (size_t)B) != cudaSuccess) {
            cudaGetLastError();
            if (M->hx) cudaFree(M->hx);
            if (M->hc) cudaFree(M->hc);
            if (M->he) cudaFree(M->he);
            M->hx = M->hc = M->he = nullptr;
            return NQS_ENOMEM;
        }
        M->h_rows = (size_t)B;
    }
    cudaStream_t st = M->h_stream;
    void *d_x = M->hx, *d_c = counts_host ? M->hc : nullptr, *d_e = M->he;
    rc = NQS_ECUDA;
    if (cudaMemcpyAsync(d_x, samples_host, 16 * (size_t)B, cudaMemcpyHostToDevice, st) == cudaSuccess &&
        (!counts_host || cudaMemcpyAsync(d_c, counts_host, 8 * (size_t)B, cudaMemcpyHostToDevice, st) == cudaSuccess)) {
        rc = nqs_local_energy(H, M, (const uint64_t *)d_x, (const int64_t *)d_c, B, minibatch, path, (float *)d_e,
                              stats_out_host, st);
        if (rc == NQS_OK) {
            if (cudaMemcpyAsync(eloc_out_host, d_e, 8 * (size_t)B, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess) rc = NQS_ECUDA;
        }
    }
    if (rc == NQS_ECUDA) cudaGetLastError();
    return rc;
}

extern "C" int64_t nqs_kernel_launch_count(void) { return g_launch_count; }

extern "C" int nqs_last_chain_kernel_ms(const nqs_made_t *M, float *ms, int *n_launches) {
    if (!M || !ms) return NQS_EINVAL;
    float total = 0.f;
    for (int b = 0; b < M->ev_used; ++b) {
        float t = 0.f;
        CU(cudaEventSynchronize(M->ev[2 * b + 1]));
        CU(cudaEventElapsedTime(&t, M->ev[2 * b], M->ev[2 * b + 1]));
        total += t;
    }
    *ms = total;
    if (n_launches) *n_launches = M->ev_used;
    return NQS_OK;
}

extern "C" const char *nqs_strerror(int status) {
    switch (status) {
        case NQS_OK: return "ok";
        case NQS_EINVAL: return "invalid argument";
        case NQS_ERANGE: return "argument out of range";
        case NQS_ENOMEM: return "out of memory";
        case NQS_ECUDA: return "CUDA error (no usable device, or a runtime call / kernel launch failed)";
        case NQS_EARCH: return "device is not compute capability 10.x (sm_100a kernels only)";
        case NQS_EUNSUPPORTED: return "requested path does not support this shape";
        default: return "unknown status";
    }
}
