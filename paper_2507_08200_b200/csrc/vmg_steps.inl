// vmg_steps.inl -- introspection and single-step entry points (include/vmg.h, second half).  Each stages the
// caller's unpadded arrays through the level's own padded arrays and runs the same kernels vmg_solve runs.

namespace {

// caller array (public layout) -> level array (internal layout) and back
int stage_in(vmg_s* h, const VmgLevel& L, double* dst, const double* src)
{
    to_internal_kernel<<<conv_grid(L.n), kThreads, 0, h->stream>>>(L.G, src, dst, nullptr);
    CUDA_TRY(h, cudaGetLastError());
    return VMG_OK;
}

int stage_out(vmg_s* h, const VmgLevel& L, double* dst, const double* src)
{
    to_natural_kernel<<<conv_grid(L.n), kThreads, 0, h->stream>>>(L.G, src, dst);
    CUDA_TRY(h, cudaGetLastError());
    return VMG_OK;
}

int finish(vmg_s* h)
{
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return VMG_OK;
}

bool bad_level(vmg_s* h, int level) { return !h || level < 0 || level >= h->nlev; }

}  // namespace

extern "C" {

int vmg_debug_pad_check(vmg_handle h, long long* nonzero)
{
    if (!h || !nonzero) return VMG_ERR_ARG;
    unsigned long long* cnt = (unsigned long long*)h->d_scal + 9;
    CUDA_TRY(h, cudaMemsetAsync(cnt, 0, sizeof(unsigned long long), h->stream));
    for (int l = 0; l < h->nlev; ++l) {
        VmgLevel& L = h->lev[l];
        const double* arrs[8] = {L.wx, L.wy, L.wz, L.dinv, L.dbase, L.phi, L.rhs, L.phi2};
        for (const double* a : arrs)
            pad_check_kernel<<<std::min<unsigned>(grid_for(L.nalloc + 2 * L.pad), 4u * h->num_sms), kThreads, 0, h->stream>>>(L.G, a, L.pad, cnt);
    }
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaMemcpyAsync(h->h_scal + 9, cnt, sizeof(unsigned long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    *nonzero = (long long)*(unsigned long long*)(h->h_scal + 9);
    return VMG_OK;
}

int vmg_num_levels(vmg_handle h) { return h ? h->nlev : VMG_ERR_ARG; }

int vmg_level_dims(vmg_handle h, int level, int dims[3])
{
    if (bad_level(h, level) || !dims) return VMG_ERR_ARG;
    dims[0] = h->lev[level].nx; dims[1] = h->lev[level].ny; dims[2] = h->lev[level].nz;
    return VMG_OK;
}

int vmg_get_level_coeffs(vmg_handle h, int level, double* a, double* bx, double* by, double* bz)
{
    if (bad_level(h, level) || level == 0 || !h->have_coeffs) return VMG_ERR_ARG;   // level 0 = the caller's own arrays
    VmgLevel& L = h->lev[level];
    if (a)  CUDA_TRY(h, cudaMemcpyAsync(a, L.a, L.n * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    if (bx) CUDA_TRY(h, cudaMemcpyAsync(bx, L.bx, face_count(L, 0) * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    if (by) CUDA_TRY(h, cudaMemcpyAsync(by, L.by, face_count(L, 1) * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    if (bz && h->three_d)
        CUDA_TRY(h, cudaMemcpyAsync(bz, L.bz, face_count(L, 2) * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    return finish(h);
}

int vmg_step_fold_bc(vmg_handle h, const double* rhs, double* btilde)
{
    if (!rhs || !btilde) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    rc = enqueue_fold_bc(h, rhs, btilde, true);
    if (rc != VMG_OK) return rc;
    return finish(h);
}

int vmg_step_smooth(vmg_handle h, int level, double* phi, const double* rhs, int nsweeps)
{
    if (bad_level(h, level) || !phi || !rhs || nsweeps < 0) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    VmgLevel& L = h->lev[level];
    if ((rc = stage_in(h, L, L.phi, phi)) != VMG_OK) return rc;
    if ((rc = stage_in(h, L, L.rhs, rhs)) != VMG_OK) return rc;
    long long count = 0;
    prepare_blocked(h);
    enqueue_smooth(h, level, nsweeps, &count);
    if ((rc = stage_out(h, L, phi, L.phi)) != VMG_OK) return rc;
    return finish(h);
}

int vmg_step_residual(vmg_handle h, int level, const double* phi, const double* rhs, double* r)
{
    if (bad_level(h, level) || !phi || !rhs || !r) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    VmgLevel& L = h->lev[level];
    if ((rc = stage_in(h, L, L.phi, phi)) != VMG_OK) return rc;
    if ((rc = stage_in(h, L, L.rhs, rhs)) != VMG_OK) return rc;
    residual_kernel<<<grid_for(L.n), kThreads, 0, h->stream>>>(view(L), L.phi, L.rhs, r);
    return finish(h);
}

int vmg_step_residual_restrict(vmg_handle h, int level, const double* phi, const double* rhs, double* rhs_coarse)
{
    if (bad_level(h, level) || level + 1 >= h->nlev || !phi || !rhs || !rhs_coarse) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    VmgLevel& L = h->lev[level];
    if ((rc = stage_in(h, L, L.phi, phi)) != VMG_OK) return rc;
    if ((rc = stage_in(h, L, L.rhs, rhs)) != VMG_OK) return rc;
    long long count = 0;
    L.cur = 0;
    plain_residual_restrict(h, level, &count);
    if ((rc = stage_out(h, h->lev[level + 1], rhs_coarse, h->lev[level + 1].rhs)) != VMG_OK) return rc;
    return finish(h);
}

int vmg_step_prolong_correct(vmg_handle h, int level, double* phi, const double* e_coarse)
{
    if (bad_level(h, level) || level + 1 >= h->nlev || !phi || !e_coarse) return VMG_ERR_ARG;
    VmgLevel& L = h->lev[level];
    int rc;
    if ((rc = stage_in(h, L, L.phi, phi)) != VMG_OK) return rc;
    if ((rc = stage_in(h, h->lev[level + 1], h->lev[level + 1].phi, e_coarse)) != VMG_OK) return rc;
    long long count = 0;
    L.cur = 0; h->lev[level + 1].cur = 0;
    plain_prolong_correct(h, level, &count);
    if ((rc = stage_out(h, L, phi, L.phi)) != VMG_OK) return rc;
    return finish(h);
}

int vmg_step_down(vmg_handle h, int level, double* phi, const double* rhs, double* rhs_coarse)
{
    if (bad_level(h, level) || level + 1 >= h->nlev || !phi || !rhs || !rhs_coarse) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    VmgLevel& L = h->lev[level];
    VmgLevel& C = h->lev[level + 1];
    if ((rc = stage_in(h, L, L.phi, phi)) != VMG_OK) return rc;
    if ((rc = stage_in(h, L, L.rhs, rhs)) != VMG_OK) return rc;
    prepare_blocked(h);
    long long count = 0;
    L.cur = 0;
    enqueue_down(h, level, &count);
    if ((rc = stage_out(h, L, phi, cur_phi(L))) != VMG_OK) return rc;
    if ((rc = stage_out(h, C, rhs_coarse, C.rhs)) != VMG_OK) return rc;
    L.cur = 0;
    return finish(h);
}

int vmg_step_up(vmg_handle h, int level, double* phi, const double* rhs, const double* e_coarse)
{
    if (bad_level(h, level) || level + 1 >= h->nlev || !phi || !rhs || !e_coarse) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    VmgLevel& L = h->lev[level];
    VmgLevel& C = h->lev[level + 1];
    if ((rc = stage_in(h, L, L.phi, phi)) != VMG_OK) return rc;
    if ((rc = stage_in(h, L, L.rhs, rhs)) != VMG_OK) return rc;
    if ((rc = stage_in(h, C, C.phi, e_coarse)) != VMG_OK) return rc;
    prepare_blocked(h);
    long long count = 0;
    L.cur = 0; C.cur = 0;
    enqueue_up(h, level, nullptr, &count);
    if ((rc = stage_out(h, L, phi, cur_phi(L))) != VMG_OK) return rc;
    L.cur = 0;
    return finish(h);
}

int vmg_step_vcycle(vmg_handle h, double* phi, const double* btilde)
{
    if (!h || !phi || !btilde) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    VmgLevel& L = h->lev[0];
    if ((rc = stage_in(h, L, L.phi, phi)) != VMG_OK) return rc;
    if ((rc = stage_in(h, L, L.rhs, btilde)) != VMG_OK) return rc;
    h->launches = 0;
    rc = run_vcycle_with_norm(h, (unsigned long long*)h->d_scal + 1);
    if (rc != VMG_OK) return rc;
    if ((rc = stage_out(h, L, phi, L.phi)) != VMG_OK) return rc;
    return finish(h);
}

int vmg_step_norm_inf(vmg_handle h, const double* v, long long n, double* out)
{
    if (!h || !v || n < 0 || !out) return VMG_ERR_ARG;
    unsigned long long* scal = (unsigned long long*)h->d_scal + 2;
    CUDA_TRY(h, cudaMemsetAsync(scal, 0, sizeof(double), h->stream));
    if (n > 0)
        norm_inf_kernel<<<std::min<unsigned>(grid_for(n), 4u * h->num_sms), kThreads, 0, h->stream>>>(v, n, scal);
    CUDA_TRY(h, cudaMemcpyAsync(h->h_scal + 2, scal, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    int rc = finish(h);
    *out = h->h_scal[2];
    return rc;
}

}  // extern "C"
