"""Host-side logic of bench.py that needs no GPU: the replicas-only aggregation over ranks (gloo, world_size 2),
per-rank seeding, the algorithmic byte count and the reference arm's JSON contract."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)
# rank 0 is the slow one in the device-timed leg, rank 1 in the e2e leg
ms = [10.0, 4.0][rank]; e2e_s = [1.0, 3.0][rank]
agg = bench.aggregate_over_ranks(ms, e2e_s, 1000.0 * (rank + 1), 10.0 * (rank + 1), 0.5e-9, world, "cpu")
w, _ = bench.make_workload("cfg2", rank)
agg["seed_probe"] = float(w.m0[0, 0, 0, 0, 0])
dist.barrier()
print("AGG" + json.dumps(agg), flush=True)
dist.destroy_process_group()
"""


def test_aggregate_over_two_ranks_gloo():
    port = _free_port()
    code = _WORKER.format(root=ROOT, port=port)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads([ln for ln in o.splitlines() if ln.startswith("AGG")][0][3:]))
    for a in outs:                                   # every rank sees the same whole-job numbers
        assert a["ms_max"] == 10.0 and a["e2e_s_max"] == 3.0          # MAX over ranks, per leg
        assert a["units"] == 3000.0 and a["e2e_units"] == 30.0        # SUM over ranks
        assert a["value"] == pytest.approx(3000.0 / 10.0e-3)
        assert a["e2e_value"] == pytest.approx(30.0 / 3.0)
        assert a["sim_t_sum"] == pytest.approx(1.0e-9)
    assert outs[0]["seed_probe"] != outs[1]["seed_probe"]            # replicas are different simulations


def test_single_rank_aggregate_is_identity():
    a = bench.aggregate_over_ranks(2.0, 0.5, 100.0, 10.0, 1e-9, 1, "cpu")
    assert a["value"] == pytest.approx(100.0 / 2e-3) and a["e2e_value"] == pytest.approx(20.0)


def test_algorithmic_bytes_match_design_table():
    # DESIGN.md 5.1 / SURVEY.md 8(d): (111 n_sub + 6 N) sizeof(T) per cell per step
    assert bench.algorithmic_bytes_per_cell_step(8, 1, 4) == 636        # cfg3: 106 B per cell-stage
    assert bench.algorithmic_bytes_per_cell_step(32, 1, 4) == 1212      # cfg5: 202
    assert bench.algorithmic_bytes_per_cell_step(1, 2, 4) == 912        # cfg4 fp32: 152
    assert bench.algorithmic_bytes_per_cell_step(1, 2, 8) == 1824       # cfg4 fp64: 304
    assert bench.algorithmic_bytes_per_cell_step(2, 1, 4) == 492        # cfg2 fp32: 82


def test_dipolar_chain_byte_count_matches_design():
    """859 MB for the FFT-convolution chain of one evaluation on CFG3 in fp32 (gather 126, R2C 202, z
    convolution with the tensor octant 255, C2R 202, scatter 50, the field read by the stage kernel 25), counted from the
    array sizes - a fixed yardstick that does not follow the implementation."""
    w, prec = bench.make_workload("cfg3_demag")
    b = bench.demag_bytes_per_evaluation(w, 4)
    nc, real2, cplx2 = 256 * 256 * 32, 512 * 512 * 32, 32 * 512 * 257
    octant = 6 * 33 * 257 * 257
    assert b == 4 * ((3 * nc + 3 * real2) + (3 * real2 + 6 * cplx2) + (12 * cplx2 + octant) + (6 * cplx2 + 3 * real2) + 6 * nc + 3 * nc)
    assert abs(b / 1e6 - 859.2) < 0.1
    r = bench.roofline_of("cfg3_demag", w, prec, 2.19 * 10, 10)
    assert r["bound"] == "hbm" and abs(r["algorithmic_bytes_per_launch"] / 1e6 - 1081.5) < 0.5 and 0.3 < r["frac"] < 0.6


def test_reference_arm_prints_one_contract_line():
    """bench.py --impl reference: the oracle on the host cores, one JSON line with the base contract's keys."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg2",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == bench.METRIC and d["unit"] == bench.UNIT
    assert d["value"] > 0 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert d["config"]["workload"] == "cfg2" and d["gpu_launches"] == 0


def test_both_arms_describe_the_workload_with_the_same_config():
    """`config` names the workload only, identically in the CUDA arm and the --impl reference arm; what differs between
    the arms (kernel path, launch mode, the oracle's bounded sample) is reported under `impl_config`."""
    w, prec = bench.make_workload("cfg2")
    cfg = bench.config_of(w, prec, "cfg2", 1)
    assert cfg["workload"] == "cfg2" and cfg["parallelism"] == "replicas x1 (no collective)"
    for key in ("kernel_path", "launch_mode", "stage_overlap", "serpentine", "reference_sample"):
        assert key not in cfg
    r = bench.roofline_of("cfg3", *bench.make_workload("cfg3")[:1], "f32", 0.2344 * 20, 20)
    assert r["bound"] == "hbm" and abs(r["algorithmic_bytes_per_launch"] - 106 * 2097152) < 1 and 0.5 < r["frac"] < 1.2
