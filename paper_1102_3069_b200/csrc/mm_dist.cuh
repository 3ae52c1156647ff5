// mm_dist.cuh -- slab decomposition over several GPUs: the partition rule, the
// per-rank context and the three compute phases between which the caller runs the two all-to-alls and the halo
// exchange.  Included by mm_api.cu (it needs mm_ctx).  Product code; shares nothing with oracle/.
//
// Layouts (float2 elements; Nzl = z1 - z0 local planes, W(p) = columns of rank p):
//   (W(p) below is the row stride: the column count rounded up to a multiple of 8)
//   slab_buf    [peer][3][Nzl][Py][W(peer)]   written by the forward y pass / read by the inverse y pass, one
//                                             launch per peer with that peer's column range (ff::ColTile)
//   pencil_buf  [3][Nz][Py][W(rank)]          the z pass runs on it in place, K-hat holds this rank's columns
// The segment (peer, component) is contiguous in both, so an all-to-all is 3 * nranks sends and receives.
#pragma once

namespace {

mm_status slab_of(const int grid[3], const int pbc[3], int nranks, int rank, mm_slab* o)
{
    if (!grid || !pbc || !o || nranks < 1 || rank < 0 || rank >= nranks) return MM_EINVAL;
    int P[3], Cs[3];
    const mm_status ps = mm_padded_size_of(grid, pbc, P, Cs);
    if (ps != MM_OK) return ps;
    const int Nz = grid[2], tiles = (Cs[0] + 15) / 16;
    if (nranks > Nz || nranks > tiles) return MM_EINVAL;
    o->rank = rank; o->nranks = nranks;
    o->z0 = (int)((long long)rank * Nz / nranks);
    o->z1 = (int)((long long)(rank + 1) * Nz / nranks);
    const int u0 = (int)((long long)rank * tiles / nranks), u1 = (int)((long long)(rank + 1) * tiles / nranks);
    o->kx0 = 16 * u0;
    o->kx1 = 16 * u1 < Cs[0] ? 16 * u1 : Cs[0];
    return MM_OK;
}

// row stride of a rank's columns in the exchange buffers: rows start on 64-byte boundaries (16-byte cp.async)
inline size_t slab_ws(const mm_slab& s) { return (size_t)((s.kx1 - s.kx0 + 7) & ~7); }

}  // namespace

extern "C" {

mm_status mm_slab_partition(const int grid[3], const int pbc[3], int nranks, int rank, mm_slab* out)
{
    return slab_of(grid, pbc, nranks, rank, out);
}

mm_status mm_create_dist(mm_ctx** out, const int grid[3], const double cellsize[3], const int pbc[3],
                         void* cuda_stream, int rank, int nranks)
{
    if (!out) return MM_EINVAL;
    *out = nullptr;
    mm_slab me;
    mm_status s = slab_of(grid, pbc, nranks, rank, &me);
    if (s != MM_OK) return fail(nullptr, s, "mm_create_dist: bad grid / rank / nranks (at most one rank per plane and per 16-column tile)");
    if (grid[2] < 2 || grid[0] % 4 != 0)
        return fail(nullptr, MM_EUNSUPPORTED, "mm_create_dist needs a 3D grid with Nx % 4 == 0");
    mm_ctx* c = nullptr;
    s = mm_create(&c, grid, cellsize, pbc, cuda_stream);
    if (s != MM_OK) return s;
    c->dist = true;
    c->slab = me;
    c->gNz = grid[2];
    c->peers.resize(nranks);
    for (int p = 0; p < nranks; ++p) slab_of(grid, pbc, nranks, p, &c->peers[p]);
    c->gmid = c->g;                         // geometry of the z pass: full lines, this rank's K-hat columns
    c->gmid.CxK = ((me.kx1 - me.kx0) + 3) & ~3;
    c->g.Nz = me.z1 - me.z0;                // every other pass and every field: the local planes
    c->g.perz = 0;                          // the ring neighbours' planes arrive as halos
    *out = c;
    return MM_OK;
}

mm_status mm_dist_buffers(mm_ctx* c, void** slab_buf, size_t* slab_elems, void** pencil_buf, size_t* pencil_elems)
{
    if (!c || !c->dist) return MM_EINVAL;
    if (!c->has_demag) return fail(c, MM_ESTATE, "mm_demag_init has not been called");
    if (slab_buf) *slab_buf = c->slab_buf;
    if (slab_elems) *slab_elems = c->slab_elems;
    if (pencil_buf) *pencil_buf = c->pencil_buf;
    if (pencil_elems) *pencil_elems = c->pencil_elems;
    return MM_OK;
}

mm_status mm_slab_segment(const int grid[3], const int pbc[3], int nranks, int rank, int peer, int comp,
                          size_t* slab_off, size_t* slab_count, size_t* pencil_off, size_t* pencil_count)
{
    mm_slab me, pr;
    mm_status s = slab_of(grid, pbc, nranks, rank, &me);
    if (s == MM_OK) s = slab_of(grid, pbc, nranks, peer, &pr);
    if (s != MM_OK) return s;
    if (comp < 0 || comp > 2) return MM_EINVAL;
    int P[3];
    mm_padded_size_of(grid, pbc, P, nullptr);
    const size_t Py = P[1], nzl = me.z1 - me.z0, Wme = slab_ws(me), Wp = slab_ws(pr), nzp = pr.z1 - pr.z0;
    size_t before = 0;                       // padded columns of the ranks below `peer`
    for (int q = 0; q < peer; ++q) {
        mm_slab t;
        slab_of(grid, pbc, nranks, q, &t);
        before += slab_ws(t);
    }
    if (slab_off) *slab_off = 3 * nzl * Py * before + (size_t)comp * nzl * Py * Wp;
    if (slab_count) *slab_count = nzl * Py * Wp;
    if (pencil_off) *pencil_off = ((size_t)comp * grid[2] + pr.z0) * Py * Wme;
    if (pencil_count) *pencil_count = nzp * Py * Wme;
    return MM_OK;
}

mm_status mm_dist_segment(const mm_ctx* c, int peer, int comp, size_t* slab_off, size_t* slab_count,
                          size_t* pencil_off, size_t* pencil_count)
{
    if (!c || !c->dist) return MM_EINVAL;
    const int grid[3] = { c->g.Nx, c->g.Ny, c->gNz };
    return mm_slab_segment(grid, c->pbc, c->slab.nranks, c->slab.rank, peer, comp, slab_off, slab_count, pencil_off,
                           pencil_count);
}

static ff::ColTile peer_tile(const mm_ctx* c, int p)
{
    ff::ColTile ct;
    const size_t W = slab_ws(c->peers[p]);
    ct.kx0 = c->peers[p].kx0; ct.ncol = c->peers[p].kx1 - c->peers[p].kx0;
    ct.a_row = c->g.CxS; ct.a_plane = (size_t)c->g.Ny * c->g.CxS;
    ct.b_row = W; ct.b_plane = (size_t)c->g.Py * W;
    return ct;
}

static mm_status dist_ready(mm_ctx* c)
{
    if (!c || !c->dist) return MM_EINVAL;
    return check_ready(c);
}

mm_status mm_dist_forward(mm_ctx* c, const float* m_slab_dev)
{
    mm_status s = dist_ready(c);
    if (s != MM_OK) return s;
    if (!m_slab_dev) return fail(c, MM_EINVAL, "NULL device pointer");
    if (!fast_fwd_x(c->fp, c->g, c->stream, m_slab_dev, c->specA)) return fail(c, MM_ECUDA, "forward x pass failed");
    c->kt.launches++;
    for (int p = 0; p < c->slab.nranks; ++p) {
        size_t off = 0;
        mm_dist_segment(c, p, 0, &off, nullptr, nullptr, nullptr);
        const ff::ColTile ct = peer_tile(c, p);
        if (!fast_y(c->fp, c->g, c->stream, -1, ct, c->specA + ct.kx0, c->slab_buf + off))
            return fail(c, MM_ECUDA, "forward y pass failed");
        c->kt.launches++;
    }
    CUDA_TRY(c, cudaGetLastError());
    return MM_OK;
}

mm_status mm_dist_mid(mm_ctx* c)
{
    mm_status s = dist_ready(c);
    if (s != MM_OK) return s;
    ff::ColTile ct;
    const size_t W = slab_ws(c->slab);
    ct.kx0 = 0; ct.ncol = c->slab.kx1 - c->slab.kx0;
    ct.a_row = 0; ct.a_plane = 0;
    ct.b_row = W; ct.b_plane = (size_t)c->g.Py * W;
    if (!fast_mid3(c->fp, c->gmid, c->stream, ct, c->pencil_buf, c->khat)) return fail(c, MM_ECUDA, "z pass failed");
    c->kt.launches++;
    CUDA_TRY(c, cudaGetLastError());
    return MM_OK;
}

mm_status mm_dist_backward(mm_ctx* c, const float* m_slab_dev, const float* halo_lo_dev, const float* halo_hi_dev,
                           float* out_slab_dev, int what, uint64_t step, double dt_th)
{
    mm_status s = dist_ready(c);
    if (s != MM_OK) return s;
    if (!out_slab_dev || what < 0 || what > 2 || (what > 0 && !m_slab_dev)) return fail(c, MM_EINVAL, "bad argument");
    for (int p = 0; p < c->slab.nranks; ++p) {
        size_t off = 0;
        mm_dist_segment(c, p, 0, &off, nullptr, nullptr, nullptr);
        const ff::ColTile ct = peer_tile(c, p);
        if (!fast_y(c->fp, c->g, c->stream, 1, ct, c->specA + ct.kx0, c->slab_buf + off))
            return fail(c, MM_ECUDA, "inverse y pass failed");
        c->kt.launches++;
    }
    const float Ms = (float)c->mat.Ms;
    if (what == 0) {
        if (!fast_inv_x_h(c->fp, c->g, c->stream, c->specA, out_slab_dev, Ms)) return fail(c, MM_ECUDA, "inverse x pass failed");
        c->kt.launches++;
    } else {
        if (!fast_inv_x_h(c->fp, c->g, c->stream, c->specA, c->hfield, 1.0f)) return fail(c, MM_ECUDA, "inverse x pass failed");
        EpiParams ep;
        std::memset(&ep, 0, sizeof(ep));
        fill_material(c, ep, step, dt_th);
        ep.mode = what == 1 ? EPI_HEFF : EPI_TORQUE;
        ep.m_in = m_slab_dev;
        ep.out = out_slab_dev;
        ep.out_scale = what == 2 ? (float)(gamma0_of(c) * c->mat.Ms) : Ms;
        ep.zlo = halo_lo_dev;
        ep.zhi = halo_hi_dev;
        ep.cell0 = (unsigned long long)c->slab.z0 * c->g.Ny * c->g.Nx;
        launch_epi4(c->g, c->hfield, ep, c->stream);
        c->kt.launches += 2;
    }
    CUDA_TRY(c, cudaGetLastError());
    return MM_OK;
}


// ---- time stepping on slabs: stage `stage` of a fixed-step method, phase by phase like an evaluation ----
static mm_status dist_tableau(mm_ctx* c, mm_method method, int stage, Tableau* tab)
{
    *tab = make_tableau(method);
    if (tab->S == 0 || tab->embedded || tab->fsal || stage < 0 || stage >= tab->S)
        return fail(c, MM_EINVAL, "slab stepping takes a stage of a fixed-step method (rk1, rk2, rk3, rk4)");
    return MM_OK;
}

mm_status mm_dist_stage_input(mm_ctx* c, mm_method method, int stage, const float* m_slab_dev, const float** in_dev_out)
{
    mm_status s = dist_ready(c);
    if (s != MM_OK) return s;
    Tableau tab;
    if ((s = dist_tableau(c, method, stage, &tab)) != MM_OK) return s;
    if (!m_slab_dev || !in_dev_out) return fail(c, MM_EINVAL, "NULL pointer");
    *in_dev_out = stage == 0 ? m_slab_dev : c->ms[(stage - 1) & 1];
    return MM_OK;
}

mm_status mm_dist_backward_stage(mm_ctx* c, float* m_slab_dev, mm_method method, int stage, double dt, uint64_t step,
                                 const float* halo_lo_dev, const float* halo_hi_dev)
{
    mm_status s = dist_ready(c);
    if (s != MM_OK) return s;
    Tableau tab;
    if ((s = dist_tableau(c, method, stage, &tab)) != MM_OK) return s;
    if (!m_slab_dev || !(dt > 0)) return fail(c, MM_EINVAL, "bad m_slab_dev / dt");
    if (stage == 0) CUDA_TRY(c, cudaMemsetAsync(c->maxbits, 0, sizeof(unsigned int), c->stream));
    for (int p = 0; p < c->slab.nranks; ++p) {
        size_t off = 0;
        mm_dist_segment(c, p, 0, &off, nullptr, nullptr, nullptr);
        const ff::ColTile ct = peer_tile(c, p);
        if (!fast_y(c->fp, c->g, c->stream, 1, ct, c->specA + ct.kx0, c->slab_buf + off))
            return fail(c, MM_ECUDA, "inverse y pass failed");
        c->kt.launches++;
    }
    if (!fast_inv_x_h(c->fp, c->g, c->stream, c->specA, c->hfield, 1.0f)) return fail(c, MM_ECUDA, "inverse x pass failed");
    EpiParams ep = stage_params(c, m_slab_dev, tab, stage, dt, step, false, false);
    ep.zlo = halo_lo_dev;
    ep.zhi = halo_hi_dev;
    ep.cell0 = (unsigned long long)c->slab.z0 * c->g.Ny * c->g.Nx;
    launch_epi4(c->g, c->hfield, ep, c->stream);
    c->kt.launches += 2;
    if (stage == tab.S - 1 && ep.m_out != m_slab_dev)         // a one-stage method leaves the new state in a scratch field
        CUDA_TRY(c, cudaMemcpyAsync(m_slab_dev, ep.m_out, 3 * ncell(c->g) * sizeof(float), cudaMemcpyDeviceToDevice,
                                    c->stream));
    CUDA_TRY(c, cudaGetLastError());
    return MM_OK;
}

}  // extern "C"
