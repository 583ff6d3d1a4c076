"""CPU checks of bench.py's evidence plumbing and of the work-list marshalling (no GPU, no compute calls)."""
import json
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import bench  # noqa: E402


def test_ncu_metric_reads_units_and_filters_kernels(tmp_path):
    f = tmp_path / "raw.csv"
    f.write_text('"ID","Kernel Name","dram__bytes_read.sum","gpu__time_duration.sum","smsp__inst_executed.sum"\n'
                 '"","","Gbyte","us","inst"\n'
                 '"0","hash_items_kernel(const int *)","1.080812","204.256000","137466370.000000"\n'
                 '"1","probe_reserve_kernel(StepParams)","2.206162","403.680000","65,564,604"\n')
    assert bench.ncu_metric(f, "hash_items", "dram__bytes_read.sum") == [1.080812e9]
    assert abs(bench.ncu_metric(f, "probe", "gpu__time_duration.sum")[0] - 403.68e-6) < 1e-12
    assert bench.ncu_metric(f, "probe", "smsp__inst_executed.sum") == [65564604.0]
    assert bench.ncu_metric(f, "nothing", "dram__bytes_read.sum") == []
    assert bench.ncu_metric(f, "probe", "no_such_metric") == []


def test_committed_ncu_evidence_names_existing_exports_and_parses():
    ev = json.loads((ROOT / "profiles" / "r02_ncu_evidence.json").read_text())
    assert len(ev["csrc_sha256"]) == 64 and len(bench.source_hash()) == 64
    for k in ("k1", "k2", "k3"):
        assert (ROOT / "profiles" / ev[k]["csv"]).exists(), ev[k]["csv"]
    rd = bench.ncu_metric(ROOT / "profiles" / ev["k1"]["csv"], ev["k1"]["kernel"], "dram__bytes_read.sum")
    assert len(rd) == 1 and 0.9e9 < rd[0] < 1.4e9                 # one bulk launch over 1 GiB of tokens
    inst = bench.ncu_metric(ROOT / "profiles" / ev["k3"]["csv"], "arc_machine_wide", "smsp__inst_executed.sum")
    assert len(inst) == len(ev["k3"]["steps"]) and min(inst) > 1e6
    # the gate: evidence is quoted only while the kernel sources are the ones that were profiled
    got, note = bench.ncu_evidence()
    assert (got is not None) == (ev["csrc_sha256"] == bench.source_hash()) and isinstance(note, str)


def test_hash_items_is_the_longest_class_first_work_list():
    from paper_2606_21238_b200 import arc

    lens = np.array([0, 15, 16, 2047 * 16 + 3, 130 * 16, 5, 400 * 16, 1024 * 16, 127 * 16 + 15, 383 * 16])
    off = np.concatenate([[7], 7 + np.cumsum(lens)]).astype(np.int64)
    it = arc.hash_items(off)
    nb = lens // 16
    assert it.dtype.itemsize == 32 and len(it) == int((nb > 0).sum())
    assert it["n_blocks"].tolist() == [2047, 1024, 400, 130, 383, 1, 127]          # >= 1024, >= 384, >= 128, the rest; stable
    key_off = np.concatenate([[0], np.cumsum(nb)])
    for rec in it:
        r = int(np.flatnonzero((off[:-1] == rec["tok_off"]) & (nb == rec["n_blocks"]))[0])
        assert rec["key_off"] == key_off[r]
    assert sorted(it["key_off"].tolist()) == sorted(key_off[:-1][nb > 0].tolist())
