// cube_ooc.inl -- brick-streamed (out-of-core) statistics and the host-cube driver.  Included by cube.cu.
//
// The paper's framework is in-core by design and rules out host memory; north_star (4)
// adds cubes larger than HBM: bricks are staged through device buffers and every accumulator
// (running (n, mean, M2, min, max), histogram bins, select digit bins) lives on the device across bricks.
// The merges are the associative/commutative ones the paper relies on.

extern "C" {

int cube_ooc_begin(cube_ctx* c, int nbins, float lo, float hi, int want_median, cudaStream_t s) {
    return cube_ooc_begin_ex(c, nbins, lo, hi, want_median, 0u, s);
}

int cube_ooc_begin_ex(cube_ctx* c, int nbins, float lo, float hi, int want_median, unsigned flags, cudaStream_t s) {
    if (!c) return CUBE_EINVAL;
    float scale = 0.f;
    const bool minmax = nbins != 0 && (flags & CUBE_RANGE_MINMAX);
    if (minmax) { if (nbins < 1 || nbins > CUBE_MAX_BINS) return CUBE_EINVAL; lo = hi = 0.f; }
    else if (nbins != 0 && !hist_scale(nbins, lo, hi, &scale)) return CUBE_EINVAL;
    c->ooc_minmax = minmax ? 1 : 0;
    c->ooc_active = 1; c->ooc_sweep = 0; c->ooc_bricks = 0;
    c->ooc_nbins = nbins; c->ooc_lo = lo; c->ooc_hi = hi; c->ooc_scale = scale;
    c->ooc_want_median = want_median ? 1 : 0;
    CUBE_CUDA(c, cudaMemsetAsync(c->gout, 0, (CUBE_MAX_BINS + 2) * sizeof(unsigned long long), s));
    CUBE_CUDA(c, cudaMemsetAsync(c->gdigits, 0, kDigitBins * sizeof(unsigned long long), s));
    {   // the running record starts empty: a rank that presents no brick (empty slab) all-gathers exactly that
        ProfScope prof(c, CUBE_K_OTHER, s);
        moments_reset_kernel<<<1, 1, 0, s>>>(c->acc, c->nvox_acc, c->mom_out);
    }
    CUBE_CUDA(c, cudaGetLastError());
    return select_init(c, 0, 1, s);
}

// The bricks are read TWICE when the median is asked for, like the cube in cube_stats (8 B per voxel, DESIGN.md
// sec. 8): sweep 0 = fused pass A (moments + first select digit), sweep 1 = fused pass B (histogram + second digit +
// compaction), last digit on the candidates (a third sweep only if the bucket did not fit the buffer).  Without
// the median: one sweep, moments and histogram.
int cube_ooc_brick(cube_ctx* c, const float* d, uint64_t nvox, cudaStream_t s) {
    if (!c || !c->ooc_active || !d || nvox == 0 || nvox > (1ull << 37)) return CUBE_EINVAL;
    int rc = CUBE_OK;
    const int acc = 1;   // cube_ooc_begin has made the running record the empty one: merging into it is the identity
    if (c->ooc_sweep == 0) {
        if (c->ooc_want_median) {
            rc = launch_moments(c, d, nvox, CUBE_COARSE_HIST, acc, s, kMomCoarse, 0.f, 0.f, false, nullptr, nullptr, c->gdigits);
        } else {
            if ((rc = launch_moments(c, d, nvox, 0u, acc, s))) return rc;
            if (c->ooc_nbins > 0 && !c->ooc_minmax)
                rc = launch_hist(c, d, nvox, c->ooc_nbins, c->ooc_lo, c->ooc_hi, c->ooc_scale, s);
        }
    } else if (c->ooc_sweep == 1) {
        const int nbins = c->ooc_nbins;
        // CUBE_RANGE_MINMAX: [min, max] of the running record -- complete after sweep 0 (a sharded run has merged the
        // ranks' records by then) -- resolved on the device, as in cube_stats
        const MomentsOut* range_from = c->ooc_minmax ? c->mom_out : nullptr;
        const float* range3 = nullptr;
        if (c->ooc_minmax && !(c->ooc_want_median && nbins <= kSmemHistMaxBins)) {
            {
                ProfScope prof(c, CUBE_K_OTHER, s);
                hist_range_kernel<<<1, 1, 0, s>>>(c->mom_out, nbins, c->range3, c->gout);
            }
            CUBE_CUDA(c, cudaGetLastError());
            range3 = c->range3;
        }
        if (!c->ooc_want_median) {    // histogram over [min, max] without the median: the second sweep is its own
            rc = launch_hist(c, d, nvox, nbins, c->ooc_lo, c->ooc_hi, c->ooc_scale, s, range3);
        } else if (nbins > 0 && nbins <= kSmemHistMaxBins) {
            const size_t smem = (size_t)hist_select_smem(nbins);
            const int occ = occupancy_of(c, hist_select_kernel, kThreads, smem);
            const int grid = grid_for(c, 4, occ < kMaxCtasPerSm ? occ : kMaxCtasPerSm);
            {
                ProfScope prof(c, CUBE_K_HIST_SELECT, s);
                hist_select_kernel<<<grid, kThreads, smem, s>>>(d, nvox, nbins, c->ooc_lo, c->ooc_hi, c->ooc_scale, range_from,
                                                                c->gbins, c->gout, c->sel, c->gdigits, c->cand, nullptr);
            }
            CUBE_CUDA(c, cudaGetLastError());
        } else if (nbins > 0) {
            // window histogram + second digit in one read when the sampled plan allows it (and the automatic variant
            // is selected); else the histogram kernel and select_pass_kernel<1> read the brick one after the other
            const bool fused_big = c->bighist == 0;
            if ((rc = launch_hist(c, d, nvox, nbins, c->ooc_lo, c->ooc_hi, c->ooc_scale, s, range3, fused_big, false))) return rc;
            rc = launch_select_pass<1>(c, d, nvox, s, nullptr, fused_big ? &c->plan->use_window : nullptr);
        } else {
            rc = launch_select_pass<1>(c, d, nvox, s);
        }
    } else if (c->ooc_sweep == 2) {
        // only the brick itself, and only if the candidates did not fit (else select_cand_kernel has counted them)
        rc = launch_select_pass<2>(c, d, nvox, s, nullptr, &c->sel->cand_done, true);
    } else {
        return CUBE_EINVAL;
    }
    c->ooc_bricks++;
    return rc;
}

// Last digit on the candidates, once per context and selection: runs iff they fitted (decided on the device).
static int ooc_count_candidates(cube_ctx* c, cudaStream_t s) {
    if (!c->cand) return CUBE_OK;
    {
        ProfScope prof(c, CUBE_K_SELECT_CAND, s);
        select_cand_kernel<<<c->num_sms, kThreads, 0, s>>>(c->sel, c->gdigits, c->cand);
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

int cube_ooc_next_sweep(cube_ctx* c, int* more, cudaStream_t s) {
    if (!c || !c->ooc_active || !more) return CUBE_EINVAL;
    int rc = CUBE_OK;
    *more = 0;
    if (!c->ooc_want_median && c->ooc_minmax) {
        *more = c->ooc_sweep == 0 ? 1 : 0;      // sweep 1: the histogram over the [min, max] found by sweep 0
        if (c->ooc_sweep > 1) return CUBE_EINVAL;
    }
    if (c->ooc_want_median) {
        if (c->ooc_sweep == 0) { rc = launch_select_scan<0>(c, c->gdigits, s); *more = 1; }
        else if (c->ooc_sweep == 1) {
            if ((rc = launch_select_scan<1>(c, c->gdigits, s))) return rc;
            if ((rc = ooc_count_candidates(c, s))) return rc;
            *more = 1;
            // Did the median's bucket fit the candidate buffer?  One 4-byte read per cube: if so the last digit
            // has just been counted on the candidates and no third sweep over the bricks is needed.
            uint32_t done = 0;
            CUBE_CUDA(c, cudaMemcpyAsync(&done, &c->sel->cand_done, sizeof(done), cudaMemcpyDeviceToHost, s));
            CUBE_CUDA(c, cudaStreamSynchronize(s));
            if (done) {
                if ((rc = launch_select_scan<2>(c, c->gdigits, s))) return rc;
                c->ooc_sweep = 2;  // becomes 3 below: result ready
                *more = 0;
            }
        }
        else if (c->ooc_sweep == 2) { rc = launch_select_scan<2>(c, c->gdigits, s); }
    }
    c->ooc_sweep++;
    return rc;
}

int cube_ooc_result(cube_ctx* c, unsigned flags, cube_moments_t* moments, uint64_t* bins, uint64_t* outside,
                    float* median, cudaStream_t s) {
    if (!c || !c->ooc_active) return CUBE_EINVAL;
    if (moments) {
        if (flags & CUBE_SAMPLE_STD) {
            // re-finalise the running partial with the sample-std denominator
            {
                ProfScope prof(c, CUBE_K_OTHER, s);
                moments_refinalize_kernel<<<1, 1, 0, s>>>(c->acc, c->nvox_acc, flags, c->mom_out);
            }
            CUBE_CUDA(c, cudaGetLastError());
        }
        CUBE_CUDA(c, cudaMemcpyAsync(moments, c->mom_out, sizeof(MomentsOut), cudaMemcpyDefault, s));
    }
    if (bins && c->ooc_nbins > 0)
        CUBE_CUDA(c, cudaMemcpyAsync(bins, c->gbins, (size_t)c->ooc_nbins * sizeof(uint64_t), cudaMemcpyDefault, s));
    if (outside && c->ooc_nbins > 0)
        CUBE_CUDA(c, cudaMemcpyAsync(outside, c->gout, 2 * sizeof(uint64_t), cudaMemcpyDefault, s));
    if (median) {
        if (!c->ooc_want_median || c->ooc_sweep < 3) return CUBE_EINVAL;
        CUBE_CUDA(c, cudaMemcpyAsync(median, &c->sel->result, sizeof(float), cudaMemcpyDefault, s));
    }
    return CUBE_OK;
}

// ---- NEXT-3: z-slab sharding over several GPUs.  The library stays free of any
// communication dependency: every rank accumulates its slab with cube_ooc_begin / cube_ooc_brick, the CALLER
// combines the exported device buffers with its collectives (NCCL through torch.distributed in
// paper_1211_4896_b200/shard.py), and cube_shard_advance runs the bucket-location kernel on the combined digit
// counts -- identical on every rank, so all ranks pick the same bucket.  No host synchronisation anywhere.
int cube_shard_buffers(cube_ctx* c, cube_shard_buffers_t* out) {
    if (!c || !out) return CUBE_EINVAL;
    out->record = c->acc;
    out->bins = reinterpret_cast<uint64_t*>(c->gbins);
    out->outside = reinterpret_cast<uint64_t*>(c->gout);
    out->digits = reinterpret_cast<uint64_t*>(c->gdigits);
    return CUBE_OK;
}

int cube_shard_merge_records(cube_ctx* c, const void* gathered, int world, unsigned flags, cudaStream_t s) {
    if (!c || !c->ooc_active || !gathered || world < 1 || world > 65536) return CUBE_EINVAL;
    {
        ProfScope prof(c, CUBE_K_OTHER, s);
        shard_merge_kernel<<<1, 1, 0, s>>>(static_cast<const unsigned char*>(gathered), world, CUBE_SHARD_RECORD_BYTES,
                                           flags & CUBE_SAMPLE_STD, c->acc, c->nvox_acc, c->mom_out);
    }
    CUBE_CUDA(c, cudaGetLastError());
    return CUBE_OK;
}

int cube_shard_advance(cube_ctx* c, int* more, cudaStream_t s) {
    if (!c || !c->ooc_active || !more) return CUBE_EINVAL;
    int rc = CUBE_OK;
    *more = 0;
    if (c->ooc_want_median) {
        if (c->ooc_sweep == 0) { rc = launch_select_scan<0>(c, c->gdigits, s); *more = 1; }
        else if (c->ooc_sweep == 1) {
            // stage 2 of this rank: its own candidates are counted here, ONCE (the scan has just cleared the digit
            // counts); the bricks presented in stage 2 are then read only if the candidates did not fit
            if ((rc = launch_select_scan<1>(c, c->gdigits, s))) return rc;
            rc = ooc_count_candidates(c, s);
            *more = 1;
        }
        else if (c->ooc_sweep == 2) { rc = launch_select_scan<2>(c, c->gdigits, s); }
        else return CUBE_EINVAL;
        c->ooc_sweep++;
    } else if (c->ooc_minmax && c->ooc_sweep == 0) {
        *more = 1;                              // stage 1: the histogram over the merged [min, max]
        c->ooc_sweep = 1;
    } else {
        c->ooc_sweep = 3;
    }
    return rc;
}

int cube_host_workspace(cube_ctx* c, size_t resident_bytes, size_t chunk_bytes) {
    if (!c) return CUBE_EINVAL;
    if (chunk_bytes == 0) chunk_bytes = (size_t)256 << 20;
    chunk_bytes = (chunk_bytes + 15) & ~(size_t)15;
    cudaFree(c->resident); c->resident = nullptr; c->resident_bytes = 0;
    cudaFree(c->chunk[0]); cudaFree(c->chunk[1]); c->chunk[0] = c->chunk[1] = nullptr;
    c->chunk_bytes = chunk_bytes;
    if (resident_bytes) {
        if (cudaMalloc(&c->resident, resident_bytes) != cudaSuccess) { cudaGetLastError(); return CUBE_ENOMEM; }
        c->resident_bytes = resident_bytes;
    }
    for (int i = 0; i < 2; ++i)
        if (cudaMalloc(&c->chunk[i], chunk_bytes) != cudaSuccess) { cudaGetLastError(); return CUBE_ENOMEM; }
    if (!c->copy_stream) {
        CUBE_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        CUBE_CUDA(c, cudaStreamCreateWithFlags(&c->work_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CUBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming));
            CUBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_consumed[i], cudaEventDisableTiming));
        }
    }
    return CUBE_OK;
}

int cube_stats_host(cube_ctx* c, const float* h, int64_t nx, int64_t ny, int64_t nz, int nbins, float lo, float hi,
                    unsigned flags, cube_moments_t* moments, uint64_t* bins, uint64_t* outside, float* median) {
    uint64_t n;
    if (!c || !h || !dims_ok(nx, ny, nz, &n)) return CUBE_EINVAL;
    if (!c->chunk[0]) {
        int rc0 = cube_host_workspace(c, 0, 0);
        if (rc0) return rc0;
    }
    const int want_median = median != nullptr;
    cudaStream_t ws = c->work_stream, cs = c->copy_stream;
    int rc = cube_ooc_begin_ex(c, (bins && outside) ? nbins : 0, lo, hi, want_median, flags & CUBE_RANGE_MINMAX, ws);
    if (rc) return rc;
    const uint64_t chunk_vox = c->chunk_bytes / sizeof(float);
    const uint64_t nchunks = (n + chunk_vox - 1) / chunk_vox;
    const bool resident = c->resident && n * sizeof(float) <= c->resident_bytes;
    int more = 1;
    for (int sweep = 0; more; ++sweep) {
        if (resident && sweep > 0) {
            // the whole cube is in HBM now: finish the select in-core, one launch per pass
            if ((rc = cube_ooc_brick(c, c->resident, n, ws))) return rc;
        } else {
            for (uint64_t i = 0; i < nchunks; ++i) {
                const uint64_t off = i * chunk_vox;
                const uint64_t cnt = (n - off < chunk_vox) ? n - off : chunk_vox;
                const int b = (int)(i & 1);
                float* dst = resident ? c->resident + off : c->chunk[b];
                if (!resident) CUBE_CUDA(c, cudaStreamWaitEvent(cs, c->ev_consumed[b], 0));
                CUBE_CUDA(c, cudaMemcpyAsync(dst, h + off, cnt * sizeof(float), cudaMemcpyHostToDevice, cs));
                CUBE_CUDA(c, cudaEventRecord(c->ev_copied[b], cs));
                CUBE_CUDA(c, cudaStreamWaitEvent(ws, c->ev_copied[b], 0));
                if ((rc = cube_ooc_brick(c, dst, cnt, ws))) return rc;
                CUBE_CUDA(c, cudaEventRecord(c->ev_consumed[b], ws));
            }
        }
        if ((rc = cube_ooc_next_sweep(c, &more, ws))) return rc;
    }
    rc = cube_ooc_result(c, flags, moments, (bins && outside) ? bins : nullptr, (bins && outside) ? outside : nullptr,
                         median, ws);
    if (rc) return rc;
    CUBE_CUDA(c, cudaStreamSynchronize(ws));
    CUBE_CUDA(c, cudaStreamSynchronize(cs));
    c->ooc_active = 0;
    return CUBE_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// Brick-callback driver: the cube never exists as a whole, neither in HBM nor in host memory (config 5).
// ------------------------------------------------------------------------------------------------
extern "C" {

int cube_stream_workspace(cube_ctx* c, size_t brick_bytes, int host_slots, size_t resident_bytes) {
    if (!c || brick_bytes == 0 || host_slots < 2 || host_slots > cube_ctx::kMaxStage) return CUBE_EINVAL;
    brick_bytes = (brick_bytes + 15) & ~(size_t)15;
    int rc = cube_host_workspace(c, resident_bytes, brick_bytes);   // device side: 2 brick buffers (+ resident)
    if (rc) return rc;
    for (int i = 0; i < cube_ctx::kMaxStage; ++i) {
        if (c->h_stage[i]) { cudaFreeHost(c->h_stage[i]); c->h_stage[i] = nullptr; }
    }
    c->stage_slots = 0; c->stage_bytes = 0;
    for (int i = 0; i < host_slots; ++i) {
        if (cudaMallocHost(&c->h_stage[i], brick_bytes) != cudaSuccess) { cudaGetLastError(); return CUBE_ENOMEM; }
        if (!c->ev_filled[i]) CUBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_filled[i], cudaEventDisableTiming));
        if (!c->ev_h2d_done[i]) CUBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_h2d_done[i], cudaEventDisableTiming));
    }
    if (!c->fill_stream) CUBE_CUDA(c, cudaStreamCreateWithFlags(&c->fill_stream, cudaStreamNonBlocking));
    c->stage_slots = host_slots; c->stage_bytes = brick_bytes;
    return CUBE_OK;
}

int cube_stats_stream(cube_ctx* c, uint64_t nbricks, uint64_t brick_vox, uint64_t total_vox, cube_fill_fn fill,
                      void* user, int nbins, float lo, float hi, unsigned flags, cube_moments_t* moments,
                      uint64_t* bins, uint64_t* outside, float* median) {
    if (!c || !fill || nbricks == 0 || brick_vox == 0 || total_vox == 0 || total_vox > (1ull << 37)) return CUBE_EINVAL;
    if ((nbricks - 1) * brick_vox >= total_vox || nbricks * brick_vox < total_vox) return CUBE_EINVAL;
    const bool want_hist = bins != nullptr || outside != nullptr;
    if (want_hist && (!bins || !outside)) return CUBE_EINVAL;
    int rc;
    if (c->stage_slots == 0 || c->stage_bytes < brick_vox * sizeof(float) || !c->chunk[0] ||
        c->chunk_bytes < brick_vox * sizeof(float)) {
        if ((rc = cube_stream_workspace(c, brick_vox * sizeof(float), 3, 0))) return rc;
    }
    const int want_median = median != nullptr;
    cudaStream_t ws = c->work_stream, cs = c->copy_stream, fs = c->fill_stream;
    if ((rc = cube_ooc_begin_ex(c, want_hist ? nbins : 0, lo, hi, want_median, flags & CUBE_RANGE_MINMAX, ws))) return rc;
    const uint64_t nres = c->resident ? (c->resident_bytes / (brick_vox * sizeof(float))) : 0;  // bricks kept in HBM
    c->stream_h2d_bytes = 0; c->stream_sweeps = 0;
    int more = 1;
    uint64_t moved = 0;   // bricks that went through the staging ring so far (slot = moved % slots, buffer = moved & 1)
    for (int sweep = 0; more; ++sweep) {
        for (uint64_t i = 0; i < nbricks; ++i) {
            const uint64_t cnt = (i + 1 == nbricks) ? total_vox - i * brick_vox : brick_vox;
            if (i < nres && sweep > 0) {                       // still in HBM from sweep 1
                if ((rc = cube_ooc_brick(c, c->resident + i * brick_vox, cnt, ws))) return rc;
                continue;
            }
            const int slot = (int)(moved % (uint64_t)c->stage_slots), b = (int)(moved & 1);
            // back-pressure: the slot's previous H2D copy must have left the staging buffer
            if (moved >= (uint64_t)c->stage_slots) CUBE_CUDA(c, cudaEventSynchronize(c->ev_h2d_done[slot]));
            if (fill(user, i, sweep, c->h_stage[slot], cnt, fs) != 0) {
                cudaDeviceSynchronize(); c->ooc_active = 0;
                return CUBE_ECALLBACK;
            }
            CUBE_CUDA(c, cudaEventRecord(c->ev_filled[slot], fs));
            float* dst = (i < nres) ? c->resident + i * brick_vox : c->chunk[b];
            CUBE_CUDA(c, cudaStreamWaitEvent(cs, c->ev_filled[slot], 0));
            if (i >= nres && moved >= 2) CUBE_CUDA(c, cudaStreamWaitEvent(cs, c->ev_consumed[b], 0));
            CUBE_CUDA(c, cudaMemcpyAsync(dst, c->h_stage[slot], cnt * sizeof(float), cudaMemcpyHostToDevice, cs));
            CUBE_CUDA(c, cudaEventRecord(c->ev_h2d_done[slot], cs));
            CUBE_CUDA(c, cudaEventRecord(c->ev_copied[b], cs));
            CUBE_CUDA(c, cudaStreamWaitEvent(ws, c->ev_copied[b], 0));
            if ((rc = cube_ooc_brick(c, dst, cnt, ws))) return rc;
            CUBE_CUDA(c, cudaEventRecord(c->ev_consumed[b], ws));
            c->stream_h2d_bytes += cnt * sizeof(float);
            ++moved;
        }
        if ((rc = cube_ooc_next_sweep(c, &more, ws))) return rc;
        c->stream_sweeps = sweep + 1;
    }
    rc = cube_ooc_result(c, flags, moments, want_hist ? bins : nullptr, want_hist ? outside : nullptr, median, ws);
    if (rc) return rc;
    CUBE_CUDA(c, cudaStreamSynchronize(ws));
    CUBE_CUDA(c, cudaStreamSynchronize(cs));
    CUBE_CUDA(c, cudaStreamSynchronize(fs));
    c->ooc_active = 0;
    return CUBE_OK;
}

int cube_stream_info(const cube_ctx* c, uint64_t* h2d_bytes, int* sweeps) {
    if (!c) return CUBE_EINVAL;
    if (h2d_bytes) *h2d_bytes = c->stream_h2d_bytes;
    if (sweeps) *sweeps = c->stream_sweeps;
    return CUBE_OK;
}

}  // extern "C"
