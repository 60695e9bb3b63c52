"""N > 1 path on the CPU: world_size-2 `gloo` processes exercise the host-side sharding logic
(SURVEY.md §8(e)): field points / matrix rows are split by `multi.my_range`, every rank evaluates its
own range against the full mesh, there is no data-path collective, and the gathered result equals
the single-process one.  The per-rank evaluation is done by the CPU oracle here (no GPU in this
tier of the tests); on a GPU box each rank calls bemcub_eval / bemcub_assemble_rows on its range
exactly the same way (bench.py)."""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, ws: int, port: int, q):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import oracle
    from paper_1606_03743_b200 import multi, synth

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=ws)
    try:
        c = synth.config1(level=1, m=101)          # 80 triangles, 101 field points: ragged split 51 / 50
        lo, hi = multi.my_range(len(c["pts"]))
        ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][lo:hi], 1)
        local = torch.as_tensor(np.concatenate([ref["phi"][:, None], ref["E"]], axis=1))
        full = multi.gather_rows(local, len(c["pts"]))
        # matrix rows shard the same way
        n = len(c["etype"])
        rlo, rhi = multi.my_range(n)
        rows, _ = oracle.assemble_rows(c["etype"], c["verts"], np.arange(rlo, rhi), oracle.default_policy(False))
        mat = multi.gather_rows(torch.as_tensor(rows), n)
        t = multi.max_over_ranks(10.0 + rank)
        u = multi.sum_over_ranks(float(hi - lo))
        # element sharding for few field points: each rank's elements, the same points, sums in rank order
        elo, ehi = multi.my_range(n)
        part = oracle.evaluate(c["etype"][elo:ehi], c["verts"][elo:ehi], c["sigma"][elo:ehi], c["pts"][:3], 1)
        tot = multi.sum_in_rank_order(torch.as_tensor(np.concatenate([part["phi"][:, None], part["E"]], axis=1))).numpy()
        dist.barrier()
        if rank == 0:
            q.put((lo, hi, full.numpy(), mat.numpy(), t, u, tot))
        else:
            assert full is None and mat is None
            q.put((lo, hi, None, None, t, u, tot))
    finally:
        dist.destroy_process_group()


def test_shard_range_covers_everything():
    from paper_1606_03743_b200 import synth
    for total in (0, 1, 7, 100, 1_000_003):
        for ws in (1, 2, 3, 8):
            edges = [synth.shard_range(total, r, ws) for r in range(ws)]
            assert edges[0][0] == 0 and edges[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
            sizes = [hi - lo for lo, hi in edges]
            assert max(sizes) - min(sizes) <= 1


@pytest.mark.timeout(180)
def test_two_rank_gloo_field_point_and_row_sharding():
    import torch.multiprocessing as mp

    import oracle
    from paper_1606_03743_b200 import synth

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=150) for _ in procs]
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    got.sort(key=lambda g: g[0])
    (lo0, hi0, full, mat, t0, u0, tot0), (lo1, hi1, _, _, t1, u1, tot1) = got
    assert (lo0, hi0, lo1, hi1) == (0, 51, 51, 101)
    assert t0 == t1 == 11.0                 # max over ranks
    assert u0 == u1 == 101.0                # whole-job units
    c = synth.config1(level=1, m=101)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], 1)
    # per-point results do not depend on how the points were sharded: bit-identical
    assert np.array_equal(full[:, 0], ref["phi"]) and np.array_equal(full[:, 1:], ref["E"])
    rows, _ = oracle.assemble_rows(c["etype"], c["verts"], np.arange(len(c["etype"])), oracle.default_policy(False))
    assert np.array_equal(mat, rows)
    # element-sharded sums: the same bits on both ranks, and the full sum up to the order of two additions
    assert np.array_equal(tot0, tot1)
    assert np.allclose(tot0[:, 0], ref["phi"][:3], rtol=1e-13, atol=0) and np.allclose(tot0[:, 1:], ref["E"][:3], rtol=1e-12, atol=1e-300)


# ------------------------------------------------------------------ the product under torch.distributed
def _gpu_worker(rank: int, ws: int, port: int, q):
    """One rank of a 2-process job sharing cuda:0: its own bemcub ctx, its contiguous range of the field
    points (bemcub_eval) and of the matrix rows (bemcub_assemble_rows), results gathered on rank 0."""
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    from paper_1606_03743_b200 import bemcub as b
    from paper_1606_03743_b200 import multi, synth

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=ws)
    try:
        c = synth.config4(scale=0.002, ntracks=23, npts_per_track=31)     # 713 field points: ragged split
        n, m = len(c["etype"]), len(c["pts"])
        with b.Context(0) as ctx:
            h = ctx.handle
            d = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda()
            b.bemcub_set_elements(h, n, d(c["etype"]), d(c["verts"]))
            lo, hi = multi.my_range(m)
            phi = torch.empty(hi - lo, dtype=torch.float64, device="cuda")
            E = torch.empty((hi - lo, 3), dtype=torch.float64, device="cuda")
            pol = b.bemcub_default_policy(True)
            b.bemcub_eval(h, d(c["sigma"]), b.RULE_ADAPTIVE, pol, hi - lo, d(c["pts"][lo:hi]), phi, E, b.F64)
            torch.cuda.synchronize()
            full = multi.gather_rows(torch.cat([phi[:, None], E], dim=1).cpu(), m)
            rlo, rhi = multi.my_range(n)
            rows = torch.empty((rhi - rlo, n), dtype=torch.float64, device="cuda")
            b.bemcub_assemble_rows(h, b.bemcub_default_policy(False), rlo, rhi - rlo, rows, n)
            torch.cuda.synchronize()
            mat = multi.gather_rows(rows.cpu(), n)
            launches = multi.sum_over_ranks(float(b.bemcub_get_stats(h)["kernel_launches"]))
            # the other sharding (few field points): this rank's contiguous range of the ELEMENTS, the same
            # five field points on every rank, per-point sums added in rank order
            elo, ehi = multi.my_range(n)
            b.bemcub_set_elements(h, ehi - elo, d(c["etype"][elo:ehi]), d(c["verts"][elo:ehi]))
            p5 = torch.empty(5, dtype=torch.float64, device="cuda")
            e5 = torch.empty((5, 3), dtype=torch.float64, device="cuda")
            b.bemcub_eval(h, d(c["sigma"][elo:ehi]), b.RULE_ADAPTIVE, pol, 5, d(c["pts"][:5]), p5, e5, b.F64)
            torch.cuda.synchronize()
            few = multi.sum_in_rank_order(torch.cat([p5[:, None], e5], dim=1).cpu())
        dist.barrier()
        q.put((rank, None if full is None else full.numpy(), None if mat is None else mat.numpy(), launches, few.numpy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.timeout(300)
def test_two_processes_one_gpu_product_path():
    """The first time two bemcub contexts run side by side under torch.distributed must not be the
    multi-GPU bench: two gloo ranks share cuda:0, each evaluates its range with the CUDA library, and
    the gathered result meets the parity bar against the oracle."""
    import torch.multiprocessing as mp

    import oracle
    from paper_1606_03743_b200 import synth

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gpu_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=240) for _ in procs], key=lambda g: g[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, full, mat, launches, few0), (_, full1, mat1, _, few1) = got
    assert full1 is None and mat1 is None and launches > 0
    c = synth.config4(scale=0.002, ntracks=23, npts_per_track=31)
    ref = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"], -1, dr=oracle.default_policy(True), want_counts=True)
    tol = np.where(ref["nana"] > 0, 1e-10, 1e-12)
    assert np.all(np.abs(full[:, 0] - ref["phi"]) <= tol * ref["Sphi"])
    assert np.all(np.abs(full[:, 1:] - ref["E"]).max(axis=1) <= tol * ref["SE"])
    A, code = oracle.assemble_rows(c["etype"], c["verts"], np.arange(len(c["etype"])), oracle.default_policy(False))
    rel = np.abs(mat - A) / np.abs(A)
    assert rel[code < 5].max() <= 1e-12 and rel[code == 5].max() <= 1e-10
    # element-sharded few-point evaluation: identical bits on both ranks, parity with the oracle's full sum
    assert np.array_equal(few0, few1)
    assert np.all(np.abs(few0[:, 0] - ref["phi"][:5]) <= tol[:5] * ref["Sphi"][:5])
    assert np.all(np.abs(few0[:, 1:] - ref["E"][:5]).max(axis=1) <= tol[:5] * ref["SE"][:5])
