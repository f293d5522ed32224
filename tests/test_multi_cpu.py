"""N > 1 plumbing on CPU: world_size-2 gloo processes exercise unit sharding, the barrier and the
max/sum-over-ranks reductions bench.py uses (the data path itself has no collective)."""
import os
import socket

import pytest
import torch.multiprocessing as mp

from paper_2511_02328_b200 import multi


def test_shard_units_partition():
    for n in (0, 1, 2, 7, 8, 1001):
        for world in (1, 2, 3, 8):
            parts = [list(multi.shard_units(n, r, world)) for r in range(world)]
            flat = [u for p in parts for u in p]
            assert flat == list(range(n))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        multi.shard_units(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r, lr, w = multi.init(backend="gloo")
    assert (r, w) == (rank, world)
    units = list(multi.shard_units(world, rank, world))
    multi.barrier()
    secs = 0.25 * (rank + 1)                      # rank 1 is the slow one
    rate, t = multi.job_throughput(100.0 * len(units), secs)
    q.put((rank, units, rate, t, multi.max_over_ranks(rank), multi.sum_over_ranks(1.0)))
    multi.finalize()


def test_gloo_world2_job_throughput():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [[0], [1]]                  # one observation per rank
    for _, _, rate, t, mx, sm in res:
        assert t == pytest.approx(0.5) and rate == pytest.approx(200.0 / 0.5)
        assert mx == 1.0 and sm == 2.0


def test_single_process_is_identity():
    assert multi.max_over_ranks(3.5) == 3.5 and multi.sum_over_ranks(2.0) == 2.0
    assert multi.env_world()[2] >= 1


# ---- ONE observation split by DM rows, one broadcast of the input, outputs stay sharded ---------
def test_shard_rows_partition():
    for ndm in (1, 2, 17, 1001):
        for world in (1, 2, 3, 8):
            got = [multi.shard_rows(ndm, r, world) for r in range(world)]
            assert got[0][0] == 0 and sum(c for _, c in got) == ndm
            for (b0, c0), (b1, _) in zip(got, got[1:]):
                assert b1 == b0 + c0


def _emu_lib():
    import ctypes
    import importlib.util
    here = os.path.dirname(os.path.abspath(__file__))
    spec = importlib.util.spec_from_file_location("build_emu", os.path.join(here, "emu", "build_emu.py"))
    build_emu = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(build_emu)
    from paper_2511_02328_b200 import binding
    lib = ctypes.CDLL(build_emu.build())
    for name, (res, args) in binding.SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    lib.ddsp_emu_faults.restype = ctypes.c_long
    lib.ddsp_emu_register.argtypes = [ctypes.c_void_p, ctypes.c_size_t]
    return lib


def _split_worker(rank, world, port, q):
    """One rank of the DM-row split.  There is no GPU here, so the rank's rows are computed by the library's
    kernels in the CPU emulation (tests/emu) through the same C ABI a GPU rank would call."""
    import ctypes
    import numpy as np
    import torch
    from paper_2511_02328_b200 import binding, synth
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    multi.init(backend="gloo")
    wl = synth.Workload("split", 9, 19, 1500.0, -6.0, 1e-3, 1700, np.linspace(0.0, 45.0, 21), mean=128.0, std=40.0)
    x = torch.zeros((wl.nchan, wl.nsamp), dtype=torch.uint8)
    if rank == 0:                                   # the ingest rank holds the observation
        x = synth.make_input(wl, "cpu")
    multi.broadcast_input(x, src=0)                 # the path's only exchange step
    begin, count = multi.shard_rows(wl.ndm, rank, world)
    lib = _emu_lib()
    dm = np.ascontiguousarray(wl.dm_list)
    h = ctypes.c_void_p()
    assert lib.ddsp_plan_create_rows(ctypes.byref(h), wl.nchan, wl.f_top, wl.chan_bw, wl.tsamp, wl.nsamp,
                                     dm.ctypes.data, dm.size, begin, count, 1, None, binding.DDSP_IN_U8) == 0
    nout = lib.ddsp_plan_nsamp_out(h)
    assert lib.ddsp_plan_set_kernel(h, binding.DDSP_KERNEL_LANES) == 0
    xin = np.ascontiguousarray(x.numpy())
    out = np.zeros((count, nout), dtype=np.uint32)
    lib.ddsp_emu_register(xin.ctypes.data, xin.nbytes)
    lib.ddsp_emu_register(out.ctypes.data, out.nbytes)
    assert lib.ddsp_execute(h, xin.ctypes.data, out.ctypes.data, None) == 0
    faults = lib.ddsp_emu_faults()
    lib.ddsp_plan_destroy(h)
    multi.barrier()
    q.put((rank, begin, count, int(nout), faults, out, xin))
    multi.finalize()


def test_gloo_world2_dm_row_split_equals_oracle(oracle):
    import numpy as np
    from paper_2511_02328_b200 import synth
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_split_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = synth.Workload("split", 9, 19, 1500.0, -6.0, 1e-3, 1700, np.linspace(0.0, 45.0, 21), mean=128.0, std=40.0)
    x = synth.make_input(wl, "cpu").numpy()
    want, nout, _ = oracle.dedisperse(x, wl.f_top, wl.chan_bw, wl.tsamp, wl.dm_list)
    assert [(r[1], r[2]) for r in res] == [(0, 11), (11, 10)]
    for rank, begin, count, nout_r, faults, out, xin in res:
        assert nout_r == nout, "every shard has the whole list's nsamp_out (d_max over all trials)"
        assert faults == 0
        assert np.array_equal(xin, x), "rank %d did not receive the broadcast input" % rank
    got = np.concatenate([r[5] for r in res], axis=0)          # outputs stay sharded; concatenated only to compare
    assert np.array_equal(got, want)
