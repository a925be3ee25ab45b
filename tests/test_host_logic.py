"""CPU-only tests: the C-ABI library loads and exports every symbol the header declares, host-side argument
checks fail loudly without a GPU, input generators, and the multi-rank statistics combine (gloo, world_size 2)."""
import ctypes
import os
import re
import socket

import numpy as np
import pytest
import torch

import paper_2112_10526_b200 as nk
from oracle import nk_oracle as orc
from paper_2112_10526_b200 import inputs as inp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as ge
    ge.build()
    return nk.load()


def test_header_and_binding_declare_the_same_symbols(lib):
    hdr = open(os.path.join(ROOT, "include", "nkb200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nk_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(nk.EXPORTS), declared ^ set(nk.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), f"{name} not exported by libnkb200.so"


def test_status_strings_and_version(lib):
    assert lib.nk_status_string(0) == b"NK_OK"
    for code in (-1, -2, -3, -4, -5):
        assert lib.nk_status_string(code).startswith(b"NK_ERR_")
    assert lib.nk_status_string(12345) == b"unknown nk_status"
    assert lib.nk_version() >= 100


def test_argument_errors_are_reported_before_any_launch(lib):
    h = ctypes.c_void_p()
    J = np.array([1.0])
    bonds = np.array([[0, 1], [1, 1]], dtype=np.int32)          # i == j: invalid
    rc = lib.nk_operator_create(ctypes.byref(h), 0, 4, 2, bonds.ctypes.data, None, 1, J.ctypes.data, 0.0, 0)
    assert rc == -1 and not h.value
    bonds = np.array([[0, 7]], dtype=np.int32)                  # out of range
    assert lib.nk_operator_create(ctypes.byref(h), 0, 4, 1, bonds.ctypes.data, None, 1, J.ctypes.data, 0.0, 0) == -1
    assert lib.nk_operator_create(ctypes.byref(h), 5, 4, 0, None, None, 1, J.ctypes.data, 0.0, 0) == -1
    assert lib.nk_rbm_logpsi_workspace_bytes(16, 10, 10, 7) == 0        # bad dtype
    assert lib.nk_rbm_logpsi_workspace_bytes(16, 10, 10, 0) > 0
    assert lib.nk_rbm_logpsi(None, 4, 10, 10, 0, None, None, None, None, None, 0, None, 0, None) == -1
    assert lib.nk_local_energy(None, None, 4, 10, 10, 0, None, None, None, 0, None, None, None, None, 0, None) == -1
    # the calls around the hot path validate on the host too (a fake non-NULL pointer is never dereferenced there)
    P = ctypes.c_void_p(256)
    assert lib.nk_local_energy_ex(None, P, 4, 10, 10, 0, P, None, None, 0, 64, P, None, None, P, 1 << 20, None) == -1
    assert lib.nk_energy_gradient_workspace_bytes(16, 10, 10, 0, 0) > 0
    assert lib.nk_energy_gradient(P, 4, 10, 10, 0, P, None, None, P, 0, None, None, P, P, 1 << 20, None) == -1  # eloc NULL
    assert lib.nk_qgt_matvec_workspace_bytes(16, 10, 10, 1, 4) > 0
    assert lib.nk_qgt_matvec(P, 4, 10, 10, 0, P, None, None, None, None, 0.0, 0, None, None, P, P, 1 << 20, None) == -1
    assert lib.nk_qgt_matvec(P, 4, 10, 10, 0, P, None, None, None, P, -1.0, 0, None, None, P, P, 1 << 20, None) == -1
    assert lib.nk_qgt_matvec(P, 4, 10, 10, 0, P, None, None, None, P, 0.0, 0, None, None, P, None, 0, None) == -3
    assert lib.nk_sr_solve_workspace_bytes(16, 10, 10, 0, 0) > lib.nk_qgt_matvec_workspace_bytes(16, 10, 10, 0, 0)
    assert lib.nk_sr_solve(P, 4, 10, 10, 0, P, None, P, P, None, 0.01, 1e-5, 10, 0, P, P, P, None, P, 1 << 20, None) == -1
    assert lib.nk_sr_solve(P, 4, 10, 10, 0, P, None, P, P, P, 0.01, -1.0, 10, 0, P, P, P, None, P, 1 << 20, None) == -1
    assert lib.nk_metropolis_workspace_bytes(1, 0, 16, 10, 10, 0, 0) == 0          # exchange rule without pairs
    assert lib.nk_metropolis_workspace_bytes(0, 0, 16, 10, 10, 0, 0) > 0
    pairs = np.array([[0, 1], [3, 10]], dtype=np.int32)                             # site 10 out of range
    assert lib.nk_metropolis_sample(1, pairs.ctypes.data, 2, P, 4, 10, 10, 0, P, None, None, 5, 0, 0, 0, 0, None, P,
                                    1 << 20, None) == -1
    assert lib.nk_metropolis_sample(7, None, 0, P, 4, 10, 10, 0, P, None, None, 5, 0, 0, 0, 0, None, P, 1 << 20, None) == -1
    assert lib.nk_metropolis_sample(0, None, 0, P, 4, 10, 10, 0, P, None, None, -1, 0, 0, 0, 0, None, P, 1 << 20, None) == -1
    assert lib.nk_rbmsymm_expand(0, 4, 10, 0, P, None, P, P, None, None) == -1
    assert lib.nk_rbmsymm_reduce_gradient(2, 4, 10, 3, P, None, P, P, None, None) == -1
    assert lib.nk_rbm_logpsi(P, 4, 10, 4097, 0, P, None, None, P, None, 0, P, 1 << 30, None) == -4               # M too large


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback_without_a_gpu(lib):
    b, c = inp.chain_bonds(4)
    with pytest.raises(nk.NkError, match="NK_ERR_CUDA"):
        nk.Operator(nk.NK_HEISENBERG, 4, b, c, [1.0])


def test_input_generators_match_the_config_table():
    sizes = {1: (10, 10, 1024, 10), 2: (100, 100, 4096, 200), 4: (100, 400, 16384, 400)}
    for c, (N, M, B, nb) in sizes.items():
        p = inp.make_config(c, n_samples=32)
        assert (p.n_sites, p.n_hidden, len(p.bonds)) == (N, M, nb)
        assert p.W.shape == (M, N) and p.sigma.shape == (32, N) and p.sigma.dtype == np.int8
        assert np.all(p.sigma.sum(axis=1) == 0) and set(np.unique(p.sigma)) == {-1, 1}
        pairs = {(min(i, j), max(i, j)) for i, j in p.bonds}
        assert len(pairs) == nb                                        # each undirected pair once
        deg = np.bincount(p.bonds.ravel(), minlength=N)
        assert np.all(deg == 2 * nb // N)
    p3 = inp.make_config(3, n_samples=8)
    assert (p3.n_sites, p3.n_hidden, len(p3.bonds), p3.h, p3.max_conn) == (400, 800, 800, 3.0, 401)
    p4 = inp.make_config(4, n_samples=8)
    assert p4.W.dtype == np.complex64 and list(p4.J) == [1.0, 0.5] and np.bincount(p4.colors).tolist() == [200, 200]
    # same seed -> same arrays; different rank offset -> different samples, same parameters
    q = inp.make_config(2, n_samples=32)
    r = inp.make_config(2, n_samples=32, sample_seed_offset=1)
    assert np.array_equal(q.W, inp.make_config(2, n_samples=4).W) and np.array_equal(q.W, r.W)
    assert not np.array_equal(q.sigma, r.sigma)


def test_combine_stats_equals_stats_of_the_union():
    rng = np.random.default_rng(0)
    e = rng.normal(size=1000) + 1j * rng.normal(size=1000)
    parts = [orc.stats(e[:100]), orc.stats(e[100:650]), orc.stats(e[650:]), (0.0, 0.0, 0.0, 0.0)]
    np.testing.assert_allclose(nk.combine_stats(parts), orc.stats(e), rtol=1e-12, atol=1e-14)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    rng = np.random.default_rng(0)
    e = rng.normal(size=1000)
    shard = e[rank::world]                                             # each rank owns a slice of the samples
    out = nk.allreduce_stats(torch.tensor(orc.stats(shard), dtype=torch.float64))
    # gradient blocks: each rank's share (1 / B_global) sum_{s in shard} O_s^* (E_s - GLOBAL mean) — what
    # nk_energy_gradient_sharded returns — for shards of unequal size; the union's force is their plain sum
    O = rng.normal(size=(1000, 7)) + 1j * rng.normal(size=(1000, 7))
    ec = e + 1j * rng.normal(size=1000)
    mine = np.arange(1000) % 3 == 0 if rank == 0 else np.arange(1000) % 3 != 0
    g_r = (np.conj(O[mine]) * (ec[mine] - ec.mean())[:, None]).sum(axis=0) / 1000.0
    g = nk.allreduce_gradient([torch.from_numpy(g_r.copy()), torch.from_numpy(g_r.real.copy())])
    q.put((rank, out.tolist(), g[0].numpy().tolist(), g[1].numpy().tolist()))
    dist.destroy_process_group()


def test_allreduce_stats_gloo_world_size_2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in procs]
    got = [q.get(timeout=120) for _ in procs]
    res = {g[0]: g[1:] for g in got}
    [p.join(60) for p in procs]
    rng = np.random.default_rng(0)
    e = rng.normal(size=1000)
    O = rng.normal(size=(1000, 7)) + 1j * rng.normal(size=(1000, 7))
    ec = e + 1j * rng.normal(size=1000)
    want = orc.force(O, ec)                                            # the unsharded force vector (Eq. (14))
    for r in range(2):
        np.testing.assert_allclose(res[r][0], orc.stats(e), rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(np.array(res[r][1]), want, atol=1e-13)
        np.testing.assert_allclose(np.array(res[r][2]), want.real, atol=1e-13)


def test_bench_gpus_flag_spawns_one_rank_per_gpu():
    """`python bench.py --gpus N` without a torchrun environment re-launches itself under torchrun with N ranks on
    127.0.0.1 (it cannot print n_gpus: 1 for --gpus 8), and a rank started with the wrong WORLD_SIZE refuses to run."""
    import argparse
    import importlib.util
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    args = argparse.Namespace(gpus=8, steps=7, warmup=3, config=5, impl="ours", no_extras=True, call="plan")
    cmd = bench.spawn_command(args, port=29511)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=8" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29511"
    tail = cmd[cmd.index(os.path.join(root, "bench.py")) + 1:]
    assert tail == ["--gpus", "8", "--steps", "7", "--warmup", "3", "--config", "5", "--impl", "ours", "--call", "plan",
                    "--no-extras"]


def test_stats_combine_c_abi_rejects_bad_arguments():
    import ctypes
    lib = nk.load()
    out = (ctypes.c_double * 4)()
    assert lib.nk_stats_combine(None, 1, out) == -1
    bad = (ctypes.c_double * 4)(0.0, 0.0, 1.0, -3.0)
    assert lib.nk_stats_combine(bad, 1, out) == -1
    assert lib.nk_stats_combine(bad, 0, out) == 0 and list(out) == [0.0, 0.0, 0.0, 0.0]
