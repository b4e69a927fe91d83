"""CPU-side checks: the C-ABI library loads and exports every symbol include/sfft.h declares (no compute
calls without a GPU), the generator is deterministic, and the N>1 sharding logic of bench.py works under
a 2-process gloo group."""
import os
import re
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sfft.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sfft_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2109_09334_b200 import binding as B
    lib = B.load_library()
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), f"libsfft_b200.so does not export {name}"
    assert sorted(B.EXPORTS) == declared, "binding.EXPORTS and include/sfft.h disagree"
    out = subprocess.run(["nm", "-D", "--defined-only", B.library_path()], capture_output=True, text=True).stdout
    for name in declared:
        assert re.search(rf"\bT {name}\b", out), name


def test_no_gpu_means_loud_failure_not_fallback():
    import torch
    from paper_2109_09334_b200 import binding as B
    assert B.sfft_strerror(B.SFFT_ERR_NOT_SPD) == "normal matrix not positive definite"
    assert "sm_100a" in B.sfft_version()
    if torch.cuda.is_available():
        return
    st, _ = B.sfft_plan_create(128, 128, 7, 1, 1, 0)
    assert st == B.SFFT_ERR_CUDA
    try:
        B.Plan(128, 128, 7, 1, 1, "poly")
    except B.SfftError as e:
        assert e.status == B.SFFT_ERR_CUDA
    else:
        raise AssertionError("Plan() must raise without a CUDA device")


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2109_09334_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "sfft_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_2109_09334_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(paper_2109_09334_b200/csrc)", "").replace("``paper_2109_09334_b200``", ""), f


def test_generator_is_deterministic_and_shaped():
    import synth
    a, b = synth.make_pair(1), synth.make_pair(1)
    assert np.array_equal(a.R, b.R) and np.array_equal(a.S, b.S)
    assert a.R.shape == (128, 128) and (a.L, a.DK, a.DB, a.basis) == (7, 1, 1, "poly")
    assert abs(np.median(a.R) - 100.0) < 3.0 and a.R.max() > 1000.0           # sky 100 ADU + stars
    c = synth.make_pair(5, subfield=3, H=64, W=64)
    d = synth.make_pair(5, subfield=4, H=64, W=64)
    assert c.basis == "bspline" and not np.array_equal(c.R, d.R)
    bt = synth.make_batch(5, nbatch=2, H=64, W=64)
    assert bt.R.shape == (2, 64, 64) and np.array_equal(bt.R[1], synth.make_pair(5, subfield=1, H=64, W=64).R)
    for k, (n, L) in {1: (150, 7), 2: (732, 11), 3: (1356, 15), 4: (1740, 17)}.items():
        cfg = synth.CONFIGS[k]
        F = (cfg["DK"] + 1) * (cfg["DK"] + 2) // 2
        assert F * cfg["L"] ** 2 + (cfg["DB"] + 1) * (cfg["DB"] + 2) // 2 == n and cfg["L"] == L


def test_shard_units_partition():
    sys.path.insert(0, ROOT)
    import bench
    for n, w in [(64, 8), (7, 2), (1, 1), (5, 8), (64, 3)]:
        parts = [bench.shard_units(n, r, w) for r in range(w)]
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(parts[i][1] == parts[i + 1][0] for i in range(w - 1))
        sizes = [hi - lo for lo, hi in parts]
        assert max(sizes) - min(sizes) <= 1


_GLOO_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
lo, hi = bench.shard_units(5, rank, 2)            # 5 independent pairs over 2 ranks, no data-path collective
mine = torch.zeros(5); mine[lo:hi] = 1.0
dist.all_reduce(mine)                             # test-only: every unit owned exactly once
# config 5 (batch of 64 sub-fields): contiguous slices of the batch axis per rank, strong scaling (SURVEY 8(e));
# the sub-fields a rank renders are exactly those of the one-process batch at its slice
import numpy as np, synth
first, cnt, scaling = bench.rank_units(5, rank, 2)
own = torch.zeros(64); own[first:first + cnt] = 1.0
dist.all_reduce(own)
assert scaling == "strong" and cnt == 32 and first == 32 * rank and torch.equal(own, torch.ones(64))
assert bench.rank_units(4, rank, 2) == (rank, 1, "weak")
part = synth.make_batch(5, nbatch=2, first=first, H=64, W=64)
assert np.array_equal(part.R[1], synth.make_pair(5, subfield=first + 1, H=64, W=64).R)
t = torch.tensor([1.0 + rank])                    # bench's max-over-ranks timing reduction
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert torch.equal(mine, torch.ones(5)) and t.item() == 2.0
dist.barrier(); dist.destroy_process_group()
print("ok", rank, lo, hi)
"""


def test_two_rank_gloo_sharding():
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    code = _GLOO_WORKER.format(root=ROOT, port=port)
    procs = [subprocess.Popen([sys.executable, "-c", code, str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
        assert o.startswith("ok")


def test_bench_configs_and_stage_names_agree_with_the_header():
    """bench.py --config accepts 1..5 and `decam` (the paper's 2046 x 4094 CCD frame, on the config-3
    recipe and model); the binding's stage list has the length include/sfft.h declares."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_2109_09334_b200 import binding as B
    assert bench.parse_config("decam") == bench.DECAM and bench.parse_config("4") == 4
    d, c3 = bench.CONFIGS[bench.DECAM], bench.CONFIGS[3]
    assert (d["H"], d["W"]) == (2046, 4094) and all(d[k] == c3[k] for k in ("L", "DK", "DB", "basis", "batch"))
    assert bench.config_dict(bench.DECAM)["unknowns"] == 1356 and "2046x4094" in bench.workload_name(bench.DECAM)
    text = open(os.path.join(ROOT, "include", "sfft.h")).read()
    assert int(re.search(r"#define SFFT_NUM_STAGES (\d+)", text).group(1)) == B.SFFT_NUM_STAGES == len(B.STAGE_NAMES)
    assert int(eval(re.search(r"#define SFFT_STATIC_MAX_PIXELS \((.*)\)", text).group(1).replace("L", ""))) == B.SFFT_STATIC_MAX_PIXELS
