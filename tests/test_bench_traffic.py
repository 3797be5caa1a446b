"""bench.py's roofline.traffic comes from profiles/traffic.csv and is valid only for the kernel sources it was captured
on: a row whose csrc hash is not the tree's yields traffic = null (no pasted constants that survive a kernel edit)."""
import argparse
import importlib.util
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

NCU_RAW = '''"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","dram__bytes_read.sum","dram__bytes_write.sum","gpu__time_duration.sum"
"","","","","","","","","","","","byte","byte","ns"
"0","1","python","box","void vr::cast_kernel<0, 0, 1, 0>(vr::FrameParams, const vr::BrickRec *)","1","7","(128, 1, 1)","(9000, 1, 1)","0","10.0","20,000,000,000","500,000,000","4300000"
"1","1","python","box","void vr::composite_kernel<0>(const vr::BrickRec *)","1","7","(256, 1, 1)","(64, 64, 1)","0","10.0","150000000","17000000","19000"
"2","1","python","box","void vr::cast_kernel<0, 0, 1, 0>(vr::FrameParams, const vr::BrickRec *)","1","7","(128, 1, 1)","(9000, 1, 1)","0","10.0","21000000000","500000000","4400000"
'''


def load_bench():
    spec = importlib.util.spec_from_file_location("bench_under_test", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_traffic_is_recorded_per_run_and_voided_by_a_kernel_edit(tmp_path, monkeypatch, capsys):
    bench = load_bench()
    monkeypatch.setattr(bench, "TRAFFIC_CSV", str(tmp_path / "traffic.csv"))
    ncu = tmp_path / "ncu.csv"
    ncu.write_text(NCU_RAW)
    args = argparse.Namespace(record_traffic=str(ncu), traffic_source="profiles/r03_cast_full.md", config=3, image=None,
                              no_skip=False)
    key = bench.traffic_key(3, 1024, 1024, 0, (2, 2, 2), True)
    assert bench.read_traffic(key)[0] is None                      # nothing captured yet
    bench.record_traffic(args)
    got, src = bench.read_traffic(key)
    assert got == (20.5e9 + 21.5e9) / 2 and "r03_cast_full" in src and "cast_kernel" in src and "2 launches" in src
    assert bench.read_traffic(bench.traffic_key(3, 1024, 1024, 0, (2, 2, 2), False))[0] is None     # another run
    bench.record_traffic(args)                                     # recording again replaces the row
    assert len(open(bench.TRAFFIC_CSV).read().strip().splitlines()) == 2
    monkeypatch.setattr(bench, "csrc_hash", lambda: "0123456789abcdef")                             # a kernel edit
    got, src = bench.read_traffic(key)
    assert got is None and "stale" in src


def test_committed_traffic_rows_are_well_formed():
    bench = load_bench()
    if not os.path.exists(bench.TRAFFIC_CSV):
        return
    import csv
    with open(bench.TRAFFIC_CSV, newline="") as f:
        rows = list(csv.DictReader(f))
    for r in rows:
        assert set(r) == set(bench.TRAFFIC_FIELDS) and float(r["bytes_per_launch"]) > 0 and len(r["csrc_sha256"]) == 16
        assert os.path.exists(os.path.join(ROOT, r["source"])), r["source"]
