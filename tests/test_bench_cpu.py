"""Host logic of bench.py that needs no GPU: the DRAM-traffic figure is a measurement read from profiles/ and is only
reported for the source tree it was captured on."""
import os
import re

import bench


def test_traffic_is_tied_to_the_source_tree():
    sha = bench.csrc_sha256()
    assert re.fullmatch(r"[0-9a-f]{64}", sha) and sha == bench.csrc_sha256()
    t, src = bench.load_traffic(12345)
    assert t is None and src["traffic_source"] is None                       # captures exist for n = 1e8 only
    t, src = bench.load_traffic(100_000_000)
    assert src["traffic_source"] and os.path.exists(os.path.join(bench.ROOT, src["traffic_source"]))
    if src.get("traffic_csrc_sha256") == sha:                                 # the capture is of this tree: a number
        assert t == src["traffic_read_bytes"] + src["traffic_write_bytes"] and 1.0e10 < t < 1.0e11
    else:                                                                      # any other tree: null and a note
        assert t is None and "stale" in src["traffic_note"]


def test_reference_arm_line_shape(capsys):
    """--impl reference times the oracle on a bounded sample and prints the contract's keys"""
    import json
    import sys
    argv = sys.argv
    sys.argv = ["bench.py", "--impl", "reference", "--steps", "1", "--warmup", "1", "--cpu-sample", "20000"]
    try:
        bench.main()
    finally:
        sys.argv = argv
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == bench.UNIT and line["higher_is_better"] is True
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"] > 0
