"""CPU checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/starkv.h declares; host-side error behaviour without a GPU; batch sharding over gloo."""
import ctypes
import importlib.util
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    spec = importlib.util.spec_from_file_location("starkv_build", os.path.join(ROOT, "paper_2606_08382_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "starkv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(starkv_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("starkv_append", "starkv_decode_attn", "starkv_pack", "starkv_unpack", "starkv_create"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_symbols(lib_path):
    import paper_2606_08382_b200 as sk
    assert sorted(sk.SYMBOLS) == declared_symbols()
    for name in sk.SYMBOLS:
        if name not in ("starkv_destroy", "starkv_last_error"):
            assert hasattr(sk, name), name


def test_strerror_and_null_handling(lib_path):
    import paper_2606_08382_b200 as sk
    assert sk.starkv_strerror(0) == "ok"
    assert "workspace" in sk.starkv_strerror(sk.STARKV_ERR_WORKSPACE)
    lib = ctypes.CDLL(lib_path)
    lib.starkv_create.restype = ctypes.c_int
    assert lib.starkv_create(None, None, None) == sk.STARKV_ERR_INVALID_ARG
    lib.starkv_page_bytes.restype = ctypes.c_size_t
    lib.starkv_page_bytes.argtypes = [ctypes.c_void_p]
    assert lib.starkv_page_bytes(None) == 0


def test_no_cpu_fallback_without_a_device(lib_path):
    """Without a CUDA device starkv_create must fail loudly (there is no CPU path)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2606_08382_b200 as sk
    with pytest.raises(sk.StarkvError) as e:
        sk.starkv_create(4, 2, 64, [16, 32], [8, 8], 64, 16, 16, 16)
    assert e.value.code == sk.STARKV_ERR_CUDA


def test_create_rejects_bad_descriptors(lib_path):
    import paper_2606_08382_b200 as sk
    bad = [
        dict(n_q_heads=5, n_kv_heads=2),                     # H_q % H_kv
        dict(rank_k=[12, 32]),                               # rank not a multiple of 8
        dict(rank_k=[16, 72]),                               # r_h > d_h
        dict(page_tokens=24),                                # page_tokens % 16
        dict(bits_hi=8, bits_lo=4, rank_k_hi=[24, 8]),       # r_hi > r
    ]
    base = dict(n_q_heads=4, n_kv_heads=2, head_dim=64, rank_k=[16, 32], rank_k_hi=[8, 8], rank_v=64,
                rank_v_hi=16, bits_hi=16, bits_lo=16, page_tokens=64)
    for b in bad:
        kw = dict(base, **b)
        with pytest.raises(sk.StarkvError) as e:
            sk.starkv_create(**kw)
        assert e.value.code == sk.STARKV_ERR_INVALID_ARG, b
    with pytest.raises(sk.StarkvError) as e:
        sk.starkv_create(**dict(base, bits_hi=4, bits_lo=3))
    assert e.value.code == sk.STARKV_ERR_UNSUPPORTED
    with pytest.raises(sk.StarkvError) as e:
        sk.starkv_create(**dict(base, layout_id=7))
    assert e.value.code == sk.STARKV_ERR_UNSUPPORTED


def test_shard_batch_partitions():
    from paper_2606_08382_b200.sharding import shard_batch
    for batch in (0, 1, 4, 7, 8, 33):
        for world in (1, 2, 3, 8):
            spans = [shard_batch(batch, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == batch
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0]
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2606_08382_b200.sharding import max_over_ranks, shard_batch
    span = shard_batch(9, rank, world)
    worst = max_over_ranks(10.0 + rank)
    q.put((rank, span, worst))
    dist.destroy_process_group()


def test_two_rank_gloo_sharding_and_max_timing():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 1000)
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == (0, 5) and res[1][1] == (5, 9)
    assert res[0][2] == res[1][2] == 11.0


def test_bench_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` times the CPU oracle (no GPU needed) and must print ONE JSON line with the contract's
    keys: same metric / unit / config as our arm, `impl`, a `cpu_baseline` describing the run and an `e2e` that repeats
    the line's value with zero copied bytes."""
    import json
    import subprocess
    import sys
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "decode_attn_latent_kv_hbm_gbs" and d["unit"] == "GB/s"
    assert d["higher_is_better"] is True and d["n_gpus"] == 1 and d["steps"] == 1 and d["vs_baseline"] is None
    assert d["config"]["workload"].startswith("C3") and d["data"] == "synthetic" and d["dtype"] == "f64"
    assert d["value"] > 0 and d["ms_per_step"] > 0
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["sample"] and cb["value"] == d["value"]
    e = d["e2e"]
    assert e["value"] == d["value"] and e["unit"] == d["unit"] and e["h2d_bytes_per_step"] == 0 and e["d2h_bytes_per_step"] == 0


def test_bench_our_arm_fails_loudly_without_a_device():
    """Our arm has no CPU fallback: without a CUDA device it must exit non-zero instead of printing a number."""
    import subprocess
    import sys
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "C3", "--steps", "1", "--warmup", "0", "--no-cpu"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode != 0
    assert not [l for l in r.stdout.strip().splitlines() if l.startswith("{") and '"value"' in l]
