"""Host-side logic of bench.py (no GPU): the flop / byte accounting of DESIGN.md sections 6-7, the step composition,
and the N > 1 path (replicas only: the one torch.distributed call is the max-over-ranks timing reduction), covered
with a world-size-2 gloo run on CPU."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_flop_convention_matches_design_section_7():
    hop = 8 * (12 + 132 + 24) - 24
    assert hop == 1320
    assert bench.flops_per_site(1, 0) == hop + 48 + 24
    assert bench.flops_per_site(1, 2) == hop + 48 + 48
    assert bench.flops_per_site(1, 1) == hop + 48 + 24 + 48
    assert bench.flops_per_site(2, 0) == 2 * hop + 240
    assert bench.flops_per_site(2, 2) == 2 * hop + 192 + 96
    assert bench.flops_per_site(2, 1) == 2 * hop + 240 + 96


def test_algorithmic_bytes_per_site_match_survey_table():
    # deg A 12-real 1152 / 576 / 296 B per site
    assert bench.bytes_per_site(1, 8, 12, 0) == 1152
    assert bench.bytes_per_site(1, 4, 12, 0) == 576
    assert bench.bytes_per_site(1, 2, 12, 0) == 296
    # xpay forms read x once more; doublets double the spinor traffic only (one link fetch for both flavors)
    assert bench.bytes_per_site(1, 8, 12, 2) == 1152 + 192
    assert bench.bytes_per_site(2, 4, 12, 0) == 8 * 12 * 4 + 2 * 96 * 2
    assert bench.bytes_per_site(2, 2, 18, 1) == 8 * 18 * 2 + 2 * 48 * 3 + 4 * 2 * 3


def test_step_composition_covers_the_metric():
    ops = bench.step_ops()
    assert len(ops) == 10
    kernels = [k for op in ops for k in bench.op_kernels(op)]
    assert len(kernels) == 20
    assert {k[1] for k in kernels if k[0] == 1} == {8, 4, 2}          # degenerate: all three precisions
    assert {k[1] for k in kernels if k[0] == 2} == {4, 2}             # non-degenerate: fp32 and half
    assert {k[2] for k in kernels} == {0, 1, 2}                       # A, A-xpay, B
    assert {k[3] for k in kernels if k[0] == 2} == {0, 1}             # plain and dagger
    vh = 32 * 32 * 32 * 64 // 2
    assert sum(bench.op_flops(o, vh) for o in ops) == 42102423552
    assert sum(bench.op_bytes(o, vh) for o in ops) == 14722007040


def test_reduce_over_ranks_is_identity_on_one_rank():
    assert bench.reduce_over_ranks(1.25, 1) == 1.25


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = bench.reduce_over_ranks(10.0 + 5.0 * rank, world)       # rank 1 is the slow replica
        q.put((rank, ms))
    finally:
        dist.destroy_process_group()


def test_replicas_timing_is_max_over_ranks_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == {0: 15.0, 1: 15.0}
    # value = N x units / max time: two replicas, the slow one sets the clock
    flops = 42102423552
    assert 2 * flops / (got[0] * 1e-3) / 1e9 == pytest.approx(2 * flops / 15e-3 / 1e9)


def test_reference_arm_other_ranks_do_no_work(monkeypatch, capsys):
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setattr(sys, "argv", ["bench.py", "--impl", "reference", "--steps", "1", "--warmup", "0"])
    bench.main()
    assert capsys.readouterr().out == ""


def test_ncu_import_ties_the_traffic_to_the_kernel_sources(tmp_path):
    """`bench.py --import-ncu`: an `ncu --page raw --csv` export (header row, units row, one row per launch) becomes the table
    bench.py reads for roofline.traffic: bytes scaled by the unit column, launches of one kernel averaged, template arguments mapped
    to the library's kernel names, and the hash of the kernel sources recorded so that a stale table reads as None."""
    src = tmp_path / "raw.csv"
    hdr = ["ID", "Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum"]
    rows = [hdr, ["", "", "Gbyte", "Mbyte", "us"],
            ["0", "void tm_dslash_generic<(int)8, (int)1, (int)12, (int)0, (bool)0, (bool)0, (bool)0>(DslashArgs)", "1.0", "200.0", "190"],
            ["1", "void tm_dslash_generic<(int)8, (int)1, (int)12, (int)0, (bool)0, (bool)0, (bool)0>(DslashArgs)", "1.2", "200.0", "190"],
            ["2", "void tm_dslash_f2<(int)2, (int)2, (int)12, (int)2, (bool)1, (bool)1, (bool)0>(DslashArgs)", "300.0", "100.0", "120"],
            ["3", "void tm_dslash_tile<(int)2, (int)1, (int)12, (int)1, (bool)0>(DslashArgs, TileGeom)", "0.25", "50.0", "70"],
            ["4", "void tm_dslash_f2<(int)4, (int)1, (int)12, (int)3, (bool)0, (bool)0, (bool)1>(DslashArgs)", "0.5", "100.0", "95"],
            ["5", "void pack_spinor_kernel<2, double>(char *)", "1", "1", "1"]]
    rows[1][2] = "Gbyte"
    rows[4][2] = "300.0"                 # this launch reported in other units below
    import csv
    with open(src, "w", newline="") as f:
        csv.writer(f, quoting=csv.QUOTE_ALL).writerows(rows)
    out = tmp_path / "traffic.csv"
    bench.import_ncu(str(src), str(out))
    h, table = bench.read_profile_table(str(out))
    assert h == bench.source_hash()
    assert table["generic<8,1,12,0,plain>"] == [1.3e9]                       # mean of (1.0 + 0.2) and (1.2 + 0.2) GB
    assert table["f2_staged<2,2,12,2,dagger>"] == [300.1e9]
    assert table["tile<2,1,12,1,plain>"] == [0.3e9]
    assert table["f2_twin<4,1,12,3,plain>"] == [0.6e9]
    assert len(table) == 4                                                  # the pack kernel is not a dslash kernel
    # a table made from other sources reads as "no traffic figure"
    stale = tmp_path / "stale.csv"
    stale.write_text(out.read_text().replace(h, "0" * 12))
    assert bench.read_profile_table(str(stale))[0] != bench.source_hash()


def test_gpus_flag_must_agree_with_the_launcher(monkeypatch):
    """`--gpus N` under torch.distributed.run must equal WORLD_SIZE (a plain `python bench.py --gpus N` starts the ranks itself)."""
    monkeypatch.setenv("WORLD_SIZE", "2")
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4"])
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert "WORLD_SIZE" in str(e.value)
