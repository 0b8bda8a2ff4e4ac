"""bench.py --gpus N runs N independent replicas (replicas only, no data-path collective);
the only cross-rank step is the max over ranks of the device-timed durations.  Covered here with two gloo ranks on
the CPU."""
import os
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist           # noqa: E402
import torch.multiprocessing as mp         # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, ms_e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 40.0 - 3.0 * rank], "cpu", world)
    out.put((rank, ms, ms_e2e, bench.whole_job_value(world, 1000, 50, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, ms_e2e, value in got:
        assert ms == 15.0 and ms_e2e == 40.0                     # the slowest rank's, on every rank
        assert value == pytest.approx(2 * 1000 * 50 / 15e-3)     # weak scaling: both replicas' units / slowest time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], "cpu", 1) == [1.5, 2.5]


def test_clock_sampler_waits_for_a_slow_nvidia_smi(tmp_path, monkeypatch):
    """The timed region of the default run lasts ~30 ms; the sampler must already deliver rows when it starts and must
    report only rows from `mark()` on (falling back to the last earlier row rather than to nothing)."""
    import os
    import stat
    import time
    import bench
    fake = tmp_path / "nvidia-smi"
    fake.write_text("#!/bin/bash\nsleep 0.4\ni=0\nwhile true; do i=$((i+1)); if [ $i -le 3 ]; then c=1000; else c=1965; fi\n"
                    "echo \"$c, 1965, 400.0, Not Active, Not Active, Not Active, Active\"; sleep 0.02; done\n")
    fake.chmod(fake.stat().st_mode | stat.S_IEXEC)
    monkeypatch.setenv("PATH", f"{tmp_path}{os.pathsep}{os.environ['PATH']}")
    s = bench.ClockSampler(0)
    assert s.rows, "constructor returns only once rows arrive"
    time.sleep(0.15)                       # "warm-up": the three 1000 MHz rows
    s.mark()
    time.sleep(0.1)
    c = s.stop()
    assert c["samples"] >= 2 and c["sm_mhz"] == 1965.0 and c["sm_max_mhz"] == 1965.0 and c["reasons"] == ["sw_power_cap"]
    s = bench.ClockSampler(0)
    s.mark()
    s.first += 1000                        # no row inside the region: the last earlier row stands in
    assert s.stop()["samples"] == 1
