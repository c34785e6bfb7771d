"""Nyquist-sampled jinc sources and the low-overhead window decomposition (the paper's distribution strategy,
PAPER.md:27-39, 386-397), on top of the batched-window solver.

The incident field, band-limited to the light cone, is represented by its samples on the lambda/2 grid, each sample
carried by one jinc source (Eq. II1).  The sources are divided into groups; each group is simulated with only the
scatterers inside the group's footprint plus a padding (an independent "window"), all windows are batched on one GPU
(or spread over GPUs as replicas: nothing is exchanged during a solve), and the scattered fields of all windows are
summed at the end.  Host-side planning only: every field / coefficient / solve runs in libtm.
"""
import numpy as np

from . import libtm


def sample_grid(k, x_range, y_range):
    """Nyquist sample coordinates x_i = i lambda/2 covering the ranges: returns (xs, ys)."""
    h = np.pi / k
    ix = np.arange(int(np.ceil(x_range[0] / h - 1e-12)), int(np.floor(x_range[1] / h + 1e-12)) + 1)
    iy = np.arange(int(np.ceil(y_range[0] / h - 1e-12)), int(np.floor(y_range[1] / h + 1e-12)) + 1)
    return ix * h, iy * h


def jinc_sources(k, x_range, y_range, z0, field_fn, drop_below=0.0):
    """Sources for a transverse field field_fn(x, y) -> (Ex, Ey) sampled on the Nyquist grid at z = z0: one jinc source per
    sample.  Returns src (S,3), the SAMPLES (S,2) complex and the grid index (S,2); the sample -> source-amplitude factor of
    the method (reading R17) is applied by the library (tm_jinc_desc.amp_is_sample), not here."""
    xs, ys = sample_grid(k, x_range, y_range)
    X, Y = np.meshgrid(xs, ys, indexing="xy")
    IX, IY = np.meshgrid(np.arange(xs.size), np.arange(ys.size), indexing="xy")
    Ex, Ey = field_fn(X.ravel(), Y.ravel())
    amp = np.stack([np.asarray(Ex, dtype=complex), np.asarray(Ey, dtype=complex)], axis=1)      # samples, not amplitudes
    src = np.stack([X.ravel(), Y.ravel(), np.full(X.size, float(z0))], axis=1)
    gi = np.stack([IX.ravel(), IY.ravel()], axis=1)
    keep = np.abs(amp).max(axis=1) > drop_below
    return src[keep], amp[keep], gi[keep]


def plan_windows(pos, src, grid_index, group, padding):
    """Divide the sources into square groups of `group` x `group` Nyquist samples; the window of a group holds the
    scatterers inside the group's bounding box grown by `padding` on every side (Fig. 2a).
    Returns a list of (source indices, scatterer indices); every source belongs to exactly one window."""
    gx, gy = grid_index[:, 0] // group, grid_index[:, 1] // group
    plans = []
    for key in sorted(set(zip(gx.tolist(), gy.tolist()))):
        sidx = np.nonzero((gx == key[0]) & (gy == key[1]))[0]
        lo = src[sidx, :2].min(axis=0) - padding
        hi = src[sidx, :2].max(axis=0) + padding
        inside = np.all((pos[:, :2] >= lo - 1e-12) & (pos[:, :2] <= hi + 1e-12), axis=1)
        plans.append((sidx, np.nonzero(inside)[0]))
    return plans


def build_batch(pos, src, amp, plans):
    """Concatenate the windows into one batched problem: positions (scatterers are duplicated where windows overlap),
    win_ptr, the global index of every batched scatterer, and the per-window source lists (src_ptr)."""
    plans = [p for p in plans if p[1].size > 0]
    scat = np.concatenate([p[1] for p in plans]) if plans else np.zeros(0, dtype=int)
    win_ptr = np.concatenate([[0], np.cumsum([p[1].size for p in plans])]).astype(np.int32)
    sord = np.concatenate([p[0] for p in plans]) if plans else np.zeros(0, dtype=int)
    src_ptr = np.concatenate([[0], np.cumsum([p[0].size for p in plans])]).astype(np.int32)
    return dict(pos=np.ascontiguousarray(pos[scat]), win_ptr=win_ptr, scat_index=scat,
                src=np.ascontiguousarray(src[sord]), amp=np.ascontiguousarray(amp[sord]), src_ptr=src_ptr)


def partition_plans(plans, rank, world):
    """Multi-GPU split: windows are independent, so rank r takes the windows r, r + world, ...; nothing is
    exchanged during the solves.  Greedy balance is unnecessary: every window holds about the same number of pairs."""
    return [p for i, p in enumerate(plans) if i % world == rank]


def sum_fields(E_local, dist=None):
    """The one communication step of the strategy ("consolidate the electric field data"): sum the detector
    fields of all ranks.  E_local: numpy complex array (M, 3); dist: an initialised torch.distributed module or None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return E_local
    import torch
    t = torch.from_numpy(np.ascontiguousarray(np.stack([E_local.real, E_local.imag], axis=0)))
    if dist.get_backend() == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    t = t.cpu().numpy()
    return t[0] + 1j * t[1]


def simulate(w, src, amp, grid_index, group, padding, pts, tol=1e-8, restart=50, max_iter=5000, precision=libtm.TM_FP64,
             stream=None, rank=0, world=1, dist=None):
    """Distributed simulation of workload `w` (global layout: pos, lmax, k, Mie radii per site or per type) driven by the
    jinc sources (src, amp = field SAMPLES as returned by jinc_sources): plan windows, batch them, solve once, sum the scattered E
    fields of all windows at `pts`.
    group = None: one window with every scatterer and every source (the undistributed reference).
    rank / world / dist: multi-GPU replicas - each rank solves its share of the windows, one all_reduce sums the fields.
    Returns (E (M,3), info dict)."""
    pos = w["pos"]
    if group is None:
        plans = [(np.arange(src.shape[0]), np.arange(pos.shape[0]))]
    else:
        plans = partition_plans(plan_windows(pos, src, grid_index, group, padding), rank, world)
    b = build_batch(pos, src, amp, plans)
    if b["pos"].shape[0] == 0:                          # a rank without windows still joins the field sum
        E = sum_fields(np.zeros((np.asarray(pts).shape[0], 3), dtype=complex), dist)
        return E, dict(n_windows=0, n_batched_scatterers=0, rc=0, iterations=0, seconds=0.0, max_rel_residual=0.0, batch=b,
                       solution=np.zeros((0, libtm.lib().tm_num_modes(w["lmax"])), dtype=complex))
    s = libtm.Solver(b["pos"], w["lmax"], w["k"], win_ptr=b["win_ptr"], precision=precision, stream=stream)
    type_of = np.asarray(w["type_of"])[b["scat_index"]]
    if w["t_kind"] in ("mie_types", "mie_sites"):
        radii = np.asarray(w["radii"])
        used, inv = np.unique(type_of, return_inverse=True)
        T = np.stack([libtm.mie_tmatrix(w["lmax"], w["k"], radii[t], w["eps_r"]) for t in used])
        s.set_tmatrices(T, inv.astype(np.int32), True, r_enclosing=radii[used])
    else:
        s.set_tmatrices(w["t_full"], type_of.astype(np.int32), False)
    s.set_incident_jinc(b["src"], b["amp"], b["src_ptr"], samples=True)
    sol, info, rc = s.solve(tol, restart, max_iter)
    E = sum_fields(s.fields(np.ascontiguousarray(pts, dtype=np.float64), sol, libtm.TM_FIELD_E_SCA), dist)
    out = dict(n_windows=len(b["win_ptr"]) - 1, n_batched_scatterers=int(b["pos"].shape[0]), rc=rc,
               iterations=max(i.iterations for i in info), seconds=info[0].seconds,
               max_rel_residual=max(i.rel_residual for i in info), batch=b, solution=sol)
    s.close()
    return E, out
