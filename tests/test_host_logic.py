"""CPU-side checks: inputs, C-ABI exports, loud failure without a GPU, generated device code on the host,
and the multi-process sharding logic (gloo, world_size 2)."""
import ctypes
import math
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import ir_eval
from paper_2510_05392_b200 import inputs
from paper_2510_05392_b200.gen import diagrams

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_rambo_inputs():
    for name in inputs.PROCESSES:
        p = inputs.momenta(name, 2000)
        assert p.shape == (2000, inputs.npar(name), 4)
        tot = p[:, 2:].sum(axis=1) - p[:, :2].sum(axis=1)
        assert np.abs(tot).max() < 1e-9                       # momentum conservation
        m = inputs.final_masses(name)
        m2 = p[:, 2:, 0] ** 2 - (p[:, 2:, 1:] ** 2).sum(-1)
        assert np.abs(m2 - m[None, :] ** 2).max() < 1e-6     # on shell
        assert (p[..., 0] > 0).all()
        # event i does not depend on the batch size (counter-based generator)
        q = inputs.momenta(name, 10, first_event=500)
        assert np.array_equal(q, p[500:510])
    assert not np.array_equal(inputs.momenta("gg_ttx", 8, seed=1), inputs.momenta("gg_ttx", 8, seed=2))


def test_library_exports_every_declared_symbol():
    """the C-ABI library loads (no GPU needed) and exports every function include/mg5_b200.h declares"""
    from paper_2510_05392_b200 import binding
    lib = binding.load_library()
    header = open(os.path.join(ROOT, "include", "mg5_b200.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(mg_[a-z0-9_]+)\s*\(", header)))
    assert declared and sorted(binding.EXPORTS) == declared
    for name in declared:
        assert hasattr(lib, name), name


@pytest.mark.skipif(os.environ.get("MG_HAVE_GPU") == "1", reason="CPU-box behaviour")
def test_no_gpu_fails_loudly():
    """without a B200 the product path raises; it never falls back to a CPU implementation"""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2510_05392_b200 import binding
    with pytest.raises(binding.MGError):
        binding.init_process("gg_ttx", "fp64")
    src = open(os.path.join(ROOT, "paper_2510_05392_b200", "binding.py")).read()
    assert "oracle" not in src.replace("CPU oracle", "")      # the binding never imports the oracle


@pytest.fixture(scope="module")
def host_jamps():
    """generated device functions + helas.cuh compiled for the host with g++ (tests only)"""
    from paper_2510_05392_b200.gen import emit_cuda
    emit_cuda.generate_all(os.path.join(ROOT, "paper_2510_05392_b200", "csrc", "generated"))
    so = os.path.join(ROOT, "tests", "_host_jamps.so")
    src = os.path.join(ROOT, "tests", "host_jamps.cpp")
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", "-o", so, src])
    lib = ctypes.CDLL(so)
    lib.host_jamps.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                               ctypes.c_void_p]
    return lib


@pytest.mark.parametrize("name,n", [("gg_ttx", 2), ("gg_ttxg", 3), ("gg_ttxgg", 4)])
def test_emitted_code_on_host_matches_ir(host_jamps, name, n):
    proc = diagrams.build_process(n)
    p = inputs.momenta(name, 3, seed=3)
    # include a beam-swapped event: externals along -z / +z
    p[2, [0, 1]] = p[2, [1, 0]]
    npar = n + 2
    for e in range(3):
        pe = np.ascontiguousarray(p[e])
        for h in range(1 << npar):
            out = np.zeros(2 * proc.ncolor)
            host_jamps.host_jamps(n, 0, pe.ctypes.data, h, inputs.PARAMS["mT"], inputs.PARAMS["wT"], out.ctypes.data)
            j = out[0::2] + 1j * out[1::2]
            hel = [1 if (h >> (npar - 1 - i)) & 1 else -1 for i in range(npar)]
            jr = ir_eval.evaluate(proc, p[e], hel, inputs.PARAMS["mT"], inputs.PARAMS["wT"])
            # external-state phases may differ per helicity but are common to all colour flows
            k = np.argmax(np.abs(jr))
            ph = (j[k] / jr[k]) / abs(j[k] / jr[k])
            assert abs(abs(ph) - 1) < 1e-12
            assert np.abs(j - ph * jr).max() < 1e-11 * np.abs(jr).max()
            if h == 5:   # float instantiation: same to single precision
                outf = np.zeros(2 * proc.ncolor)
                host_jamps.host_jamps(n, 1, pe.ctypes.data, h, inputs.PARAMS["mT"], inputs.PARAMS["wT"], outf.ctypes.data)
                jf = outf[0::2] + 1j * outf[1::2]
                assert np.abs(jf - j).max() < 2e-4 * np.abs(j).max()


def test_two_rank_sharding_gloo(tmp_path):
    """N > 1 path of bench.py on CPU (gloo, world_size 2), calling bench.py's own functions: disjoint contiguous event
    shards, the max-over-ranks reduction of the device time, and the agreement check of the helicity masks.  The masks
    themselves come from the oracle's per-helicity terms on each rank's own probe events with the 1e-8 rule of reading A5:
    a property of the process, the same on every shard."""
    script = tmp_path / "w.py"
    script.write_text(f"""
import os, sys
sys.path.insert(0, {ROOT!r})
import numpy as np, torch, torch.distributed as dist
import bench, oracle
from paper_2510_05392_b200 import inputs
dist.init_process_group('gloo')
rank, world = dist.get_rank(), dist.get_world_size()
nevt = 64
first = bench.shard_first_event(rank, nevt)
assert first == rank * nevt
mom = inputs.momenta('gg_ttx', nevt, seed=1, first_event=first)            # weak scaling: each rank its own events
full = inputs.momenta('gg_ttx', nevt * world, seed=1)
assert np.array_equal(mom, full[rank * nevt:(rank + 1) * nevt])
assert bench.reduce_max_ms(10.0 + rank, dist) == 10.0 + world - 1
for process in ('epem_mupmum', 'gg_ttxg'):
    m = inputs.momenta(process, nevt, seed=1, first_event=first)
    me, meh = oracle.matrix_elements(process, m, inputs.PARAMS, per_helicity=True)
    mask = (meh / me[:, None] > 1e-8).any(axis=0)
    assert bench.masks_agree(mask, dist), process
    bad = mask.copy(); bad[0] ^= (rank == 1)
    assert not bench.masks_agree(bad, dist)
dist.barrier()
if rank == 0:
    print('OK', world)
dist.destroy_process_group()
""")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29533", str(script)],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "OK 2" in r.stdout


def test_bench_gpus_flag_spawns_ranks_and_fails_loudly_without_gpu():
    """`python bench.py --gpus 2` starts two ranks itself; on a CPU box every rank refuses to run (no fallback)"""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"], capture_output=True,
                       text=True, timeout=300, env=env)
    assert r.returncode != 0
    # the launcher ends the other rank as soon as the first one exits, so one message is certain and a second is likely
    assert "no CPU fallback" in (r.stdout + r.stderr)
    # a world size that contradicts --gpus is an error, not a silent single-GPU run
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4"], capture_output=True, text=True,
                       timeout=120, env=dict(env, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0"))
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stdout + r.stderr)
