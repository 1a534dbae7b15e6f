// host_api.inl -- md_eri4_host / md_eri3_host: the same kernels behind host buffers.
// Inputs are staged with cudaMemcpyAsync on the caller's stream into stream-ordered
// temporaries (cudaMallocAsync), the result is copied back (overlapped with compute for large quartet
// lists), and the stream is synchronised.
namespace {

struct DeviceCopy {
    std::vector<void *> blocks;
    cudaStream_t st;
    explicit DeviceCopy(cudaStream_t s) : st(s) {}
    ~DeviceCopy() { for (void *p : blocks) cudaFreeAsync(p, st); }
    cudaError_t alloc(void **d, size_t bytes) {
        cudaError_t e = cudaMallocAsync(d, bytes ? bytes : 8, st);
        if (e == cudaSuccess) blocks.push_back(*d);
        return e;
    }
    template <class T> cudaError_t up(const T *h, size_t n, const T **d) {
        void *p = nullptr;
        cudaError_t e = alloc(&p, n * sizeof(T));
        if (e != cudaSuccess) return e;
        *d = (const T *)p;
        return n ? cudaMemcpyAsync(p, h, n * sizeof(T), cudaMemcpyHostToDevice, st) : cudaSuccess;
    }
    cudaError_t shells(const md_shells &h, md_shells *d) {
        *d = h;
        cudaError_t e;
        if ((e = up(h.center, (size_t)h.n * 3, &d->center)) != cudaSuccess) return e;
        if ((e = up(h.exps, (size_t)h.n * h.K, &d->exps)) != cudaSuccess) return e;
        return up(h.coefs, (size_t)h.n * h.K, &d->coefs);
    }
    cudaError_t pairs(const md_pairs &h, md_pairs *d) {
        *d = h;
        cudaError_t e;
        if ((e = shells(h.a, &d->a)) != cudaSuccess) return e;
        if ((e = shells(h.b, &d->b)) != cudaSuccess) return e;
        if (h.idx) return up(h.idx, (size_t)h.npairs * 2, &d->idx);
        return cudaSuccess;
    }
};

int host_call(const md_pairs *bra, const md_pairs *ket, const md_shells *X, int64_t n, const int32_t *idx, int pure,
              int layout, double *out, int64_t cap, void *stream) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = ket ? check_pairs(ket) : check_shells(X))) return e;
    if (n < 0 || (pure != 0 && pure != 1)) return MD_EINVAL;
    int64_t need = ket ? md_eri4_out_elems(bra->a.l, bra->b.l, ket->a.l, ket->b.l, pure, n)
                       : md_eri3_out_elems(bra->a.l, bra->b.l, X->l, pure, n);
    if (need < 0) return (int)need;
    if (need > cap) return MD_ECAPACITY;
    if (n > 0 && !out) return MD_EINVAL;
    if ((e = md_init())) return e;
    cudaStream_t st = (cudaStream_t)stream;
    DeviceCopy dc(st);
    md_pairs dbra, dket;
    md_shells dX;
    CK(dc.pairs(*bra, &dbra));
    if (ket) CK(dc.pairs(*ket, &dket)); else CK(dc.shells(*X, &dX));
    const int32_t *didx = nullptr;
    if (idx) CK(dc.up(idx, (size_t)n * 2, &didx));
    void *dout = nullptr;
    CK(dc.alloc(&dout, (size_t)need * 8));
    // Quartet lists in the quartet-major layout are cut into chunks: the device-to-host copy of chunk i runs on an
    // internal copy stream while the kernels of chunk i+1 run on the caller's stream.
    const int64_t per = n > 0 ? need / n : 0;
    const int nchunk = (idx && layout == MD_LAYOUT_QUARTET_MAJOR && n >= 32768) ? (int)std::min<int64_t>(8, n / 16384) : 1;
    if (nchunk <= 1) {
        e = ket ? md_eri4(&dbra, &dket, n, didx, pure, layout, (double *)dout, need, stream)
                : md_eri3(&dbra, &dX, n, didx, pure, layout, (double *)dout, need, stream);
        if (e) { cudaStreamSynchronize(st); return e; }
        CK(cudaMemcpyAsync(out, dout, (size_t)need * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        return MD_OK;
    }
    // per-call copy stream and events (no state survives the call: the function is reentrant)
    struct Copier {
        cudaStream_t s = nullptr;
        cudaEvent_t done[8] = {};
        ~Copier() {
            for (auto &ev : done) if (ev) cudaEventDestroy(ev);
            if (s) cudaStreamDestroy(s);
        }
    } cp;
    CK(cudaStreamCreateWithFlags(&cp.s, cudaStreamNonBlocking));
    for (auto &ev : cp.done) CK(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    cudaStream_t copy_stream = cp.s;
    cudaEvent_t *done = cp.done;
    for (int c = 0; c < nchunk; ++c) {
        const int64_t q0 = n * c / nchunk, q1 = n * (c + 1) / nchunk, nc = q1 - q0;
        double *dchunk = (double *)dout + q0 * per;
        e = ket ? md_eri4(&dbra, &dket, nc, didx + 2 * q0, pure, layout, dchunk, nc * per, stream)
                : md_eri3(&dbra, &dX, nc, didx + 2 * q0, pure, layout, dchunk, nc * per, stream);
        if (e) { cudaStreamSynchronize(st); cudaStreamSynchronize(copy_stream); return e; }
        CK(cudaEventRecord(done[c], st));
        CK(cudaStreamWaitEvent(copy_stream, done[c], 0));
        CK(cudaMemcpyAsync(out + q0 * per, dchunk, (size_t)(nc * per) * 8, cudaMemcpyDeviceToHost, copy_stream));
    }
    CK(cudaStreamSynchronize(copy_stream));
    CK(cudaStreamSynchronize(st));
    return MD_OK;
}

}  // namespace

extern "C" {
int md_eri4_host(const md_pairs *bra, const md_pairs *ket, int64_t nquartets, const int32_t *quartet_idx, int pure,
                 int layout, double *out, int64_t out_capacity_elems, void *cuda_stream) {
    if (!ket) return MD_EINVAL;
    return host_call(bra, ket, nullptr, nquartets, quartet_idx, pure, layout, out, out_capacity_elems, cuda_stream);
}
int md_eri3_host(const md_pairs *bra, const md_shells *X, int64_t ntriplets, const int32_t *triplet_idx, int pure,
                 int layout, double *out, int64_t out_capacity_elems, void *cuda_stream) {
    if (!X) return MD_EINVAL;
    return host_call(bra, nullptr, X, ntriplets, triplet_idx, pure, layout, out, out_capacity_elems, cuda_stream);
}
}
