"""CPU-only, world_size-2 `gloo` tests of the N > 1 path (replicas over time chunks, no collective
on the data path). What is covered without a GPU:
  * `aa_strategy_shard` (host logic inside libaa.so, on a planned strategy): rank r of W owns chunks r, r+W, ...; the
    shards tile the chunk list exactly once; a rank with no chunk is legal;
  * `replicas.gather_candidates` / `canonical_order` / `max_over_ranks` over a real 2-process gloo group: every rank
    searches ITS chunks (here with the oracle standing in for the GPU — tests may use it), the gathered list equals the
    single-process search of all chunks, in canonical order.
"""
import os
import socket
import tempfile

import numpy as np
import pytest

import datagen
import oracle
import paper_1912_07704_b200 as aa
from datagen.workloads import scaled
from paper_1912_07704_b200 import replicas


def _workload():
    w = scaled(datagen.get_workload("tiny"), nsamp=6000, name="tiny6k")
    return w


def _planned(w, chunk_len_hint):
    plan = aa.aa_plan_create(w.freqs_mhz, w.tsamp_s, w.ranges, w.widths, w.threshold)
    st = aa.aa_strategy_plan(plan, w.nsamp, chunk_len_hint=chunk_len_hint)
    return plan, st


def _oracle_chunk_candidates(w, x, k, chunk):
    start, length, n_out = chunk
    out = []
    for r, rng in enumerate(w.ranges):
        xb = oracle.bin_time(x, start, length // rng[3], rng[3])
        out.append(oracle.search_rows(xb, k, rng, r, n_out // rng[3], w.widths, w.threshold, start, 0, rng[2], want=())["cands"])
    return np.concatenate(out)


def test_shard_tiles_the_chunk_list_once():
    w = _workload()
    plan, st = _planned(w, 1024)
    try:
        n = aa.aa_strategy_get_info(st)["nchunks"]
        assert n >= 5
        for world in (1, 2, 3, n, n + 2):
            seen = []
            for rank in range(world):
                aa.aa_strategy_shard(st, rank, world)
                info = aa.aa_strategy_get_info(st)
                assert (info["shard_rank"], info["shard_world"], info["next_chunk"]) == (rank, world, rank)
                mine = replicas.chunks_of_rank(n, rank, world)
                assert mine == list(range(rank, n, world))
                seen += mine
            assert sorted(seen) == list(range(n))
        with pytest.raises(aa.AaError) as e:
            aa.aa_strategy_shard(st, 2, 2)
        assert e.value.status == aa.AA_ERR_INVALID_ARG and "rank" in e.value.message
        # a planned strategy still refuses to run, sharded or not
        with pytest.raises(aa.AaError) as e:
            aa.aa_run_sps(st)
        assert e.value.status == aa.AA_ERR_NOT_READY
    finally:
        aa.aa_strategy_destroy(st)
        aa.aa_plan_destroy(plan)


def test_input_span_of_rank_covers_only_its_chunks():
    chunks = [(0, 100, 80), (80, 100, 80), (160, 100, 80), (240, 60, 40)]
    assert replicas.input_span_of_rank(chunks, 0, 2) == (0, 260)
    assert replicas.input_span_of_rank(chunks, 1, 2) == (80, 300)
    assert replicas.input_span_of_rank(chunks, 5, 6) is None


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, outdir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload()
        pl, dms, dl = w.pulses()
        x = datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl)
        k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        plan, st = _planned(w, 1024)
        aa.aa_strategy_shard(st, rank, world)
        info = aa.aa_strategy_get_info(st)
        chunks = [aa.aa_strategy_get_chunk(st, j) for j in range(info["nchunks"])]
        mine = replicas.chunks_of_rank(len(chunks), info["shard_rank"], info["shard_world"])
        parts = [_oracle_chunk_candidates(w, x, k, chunks[j]) for j in mine]
        local = np.concatenate(parts) if parts else np.zeros(0, oracle.CAND_DTYPE)
        merged = replicas.gather_candidates(local, info["n_out"])
        slowest = replicas.max_over_ranks(1.0 + rank)
        np.save(os.path.join(outdir, f"merged{rank}.npy"), merged)
        with open(os.path.join(outdir, f"t{rank}.txt"), "w") as f:
            f.write(f"{slowest} {len(local)} {len(mine)}")
        aa.aa_strategy_destroy(st)
        aa.aa_plan_destroy(plan)
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_gather_equals_single_process_search():
    import torch.multiprocessing as mp
    world = 2
    with tempfile.TemporaryDirectory() as d:
        mp.spawn(_rank_main, args=(world, _free_port(), d), nprocs=world, join=True)
        merged = [np.load(os.path.join(d, f"merged{r}.npy")) for r in range(world)]
        times = [open(os.path.join(d, f"t{r}.txt")).read().split() for r in range(world)]
    # single process: all chunks in order
    w = _workload()
    pl, dms, dl = w.pulses()
    x = datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl)
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    g = oracle.chunk_geometry(k, w.ranges, w.nsamp, chunk_len=1024)
    exp = np.concatenate([_oracle_chunk_candidates(w, x, k, c) for c in g["chunks"]])
    assert len(exp) > 0
    for m in merged:                                     # every rank holds the same, complete, canonically ordered list
        assert m.dtype == exp.dtype and len(m) == len(exp)
        for f in exp.dtype.names:
            assert np.array_equal(m[f], exp[f]), f
    assert [float(t[0]) for t in times] == [2.0, 2.0]    # max over ranks of (1.0, 2.0)
    assert sum(int(t[1]) for t in times) == len(exp)     # the shards partition the candidates
    assert sum(int(t[2]) for t in times) == len(g["chunks"])
