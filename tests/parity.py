"""Parity harness shared by the GPU tests, smoke() and bench.py's sanity leg.

Feeds identical fp32 arrays to the CUDA path (through the C-ABI binding) and to the CPU oracle and
compares per DESIGN.md section 5 (readings S20-S22, S25):
  * integer outputs (hash, sorted_hash, perm, cell tables, comm_hash, boundary list, counts):
    bit-exact;
  * float fields drho, acc, dsig and the post-step state: max |gpu - oracle| over particles and
    components divided by max |oracle| over the same set <= tol (1e-5 for rates: BASELINE.json
    north_star; 1e-6 for the state, which is dominated by the unchanged fp32 inputs);
    an identically-zero oracle field requires |gpu| < 1e-30 (S21);
  * pair_count: relative 1e-6 (S25: fp32 vs fp64 compare at the support radius).
"""
from __future__ import annotations

import numpy as np
import torch

RATE_TOL = 1e-5
STATE_TOL = 1e-6


def field_err(gpu: np.ndarray, ref: np.ndarray) -> float:
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    assert gpu.shape == ref.shape, (gpu.shape, ref.shape)
    if ref.size == 0:
        return 0.0
    scale = np.max(np.abs(ref))
    err = np.max(np.abs(gpu - ref))
    if scale == 0.0:
        return 0.0 if err < 1e-30 else float("inf")
    return float(err / scale)


def u32(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().numpy().view(np.uint32)


def compare_integers(out, ref, n) -> None:
    """out: sph.StepOutputs (device), ref: oracle.StepResult."""
    np.testing.assert_array_equal(u32(out.hash), ref.hash, err_msg="hash")
    np.testing.assert_array_equal(u32(out.sorted_hash), ref.sorted_hash, err_msg="sorted_hash")
    np.testing.assert_array_equal(u32(out.perm), ref.perm, err_msg="perm")
    np.testing.assert_array_equal(u32(out.cell_start), ref.cell_start, err_msg="cell_start")
    np.testing.assert_array_equal(u32(out.cell_end), ref.cell_end, err_msg="cell_end")
    np.testing.assert_array_equal(u32(out.comm_hash), ref.comm_hash, err_msg="comm_hash")
    m = int(u32(out.boundary_count)[0])
    assert m == ref.boundary_ids.shape[0], ("boundary_count", m, ref.boundary_ids.shape[0])
    np.testing.assert_array_equal(u32(out.boundary_ids)[:m], ref.boundary_ids, err_msg="boundary_ids")
    np.testing.assert_array_equal(u32(out.owner_counts), ref.owner_counts, err_msg="owner_counts")


def compare_rates(out, rates, idx=None) -> dict:
    """Rates indexed by sorted position; idx selects the sampled positions the oracle computed."""
    drho = out.drho.cpu().numpy()
    acc = out.acc.cpu().numpy()
    dsig = out.dsig.cpu().numpy().T            # [n,6]
    if idx is not None:
        drho, acc, dsig = drho[idx], acc[idx], dsig[idx]
    errs = {
        "drho": field_err(drho, rates.drho),
        "acc": field_err(acc[:, :3], rates.acc),
        "dsig": field_err(dsig, rates.dsig),
    }
    assert np.all(acc[:, 3] == 0.0)
    for k, v in errs.items():
        assert v <= RATE_TOL, (k, v)
    return errs


def compare_state(state, ref) -> dict:
    errs = {
        "pos": field_err(state.posm.cpu().numpy()[:, :3], ref.posm[:, :3]),
        "mass": field_err(state.posm.cpu().numpy()[:, 3], ref.posm[:, 3]),
        "vel": field_err(state.velr.cpu().numpy()[:, :3], ref.velr[:, :3]),
        "rho": field_err(state.velr.cpu().numpy()[:, 3], ref.velr[:, 3]),
        "sig": field_err(state.sig.cpu().numpy(), ref.sig),
    }
    for k, v in errs.items():
        assert v <= STATE_TOL, (k, v)
    return errs


def lockstep(sph, oracle, w, steps=1, flags=0, floats=True, hp=None) -> list[dict]:
    """Reading S20: every step the oracle is fed the GPU's fp32 state at the start of that step.
    hp = per-particle smoothing lengths in id order (NEXT-4): sph_step_varh against oracle.step(hp=)."""
    ctx = sph.Context.for_workload(w, flags=flags)
    state = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    out = ctx.alloc_outputs(w.n)
    h_dev = torch.from_numpy(np.ascontiguousarray(hp, np.float32)).cuda() if hp is not None else None
    report = []
    for _ in range(steps):
        posm, velr = state.posm.cpu().numpy(), state.velr.cpu().numpy()
        sig, owner = state.sig.cpu().numpy(), state.owner.cpu().numpy()
        ref = oracle.step(posm, velr, sig, owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt,
                          floats=floats, hp=hp)
        if hp is None:
            ctx.sph_step(state, w.dt, out)
        else:
            ctx.sph_step_varh(state, h_dev, w.dt, out)
        torch.cuda.synchronize()
        compare_integers(out, ref, w.n)
        np.testing.assert_array_equal(state.owner.cpu().numpy(), owner)
        r = {"boundary": int(ref.boundary_ids.shape[0])}
        if floats:
            r.update(compare_rates(out, ref.rates))
            r.update(compare_state(state, ref))
            pc = int(out.pair_count.cpu()[0])
            r["pairs"] = pc
            assert abs(pc - ref.rates.pair_count) <= max(1e-6 * ref.rates.pair_count, 2), \
                (pc, ref.rates.pair_count)
        report.append(r)
    ctx.close()
    return report
