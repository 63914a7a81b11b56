"""gpfc_fold_stream (-m gpu): the chunked fold hands every
finished chunk to a consumer on another stream while the next chunk folds.  The assembled
result must equal the monolithic gpfc_fold_batch call bit for bit, whatever the chunking."""
import numpy as np
import pytest

from paper_2312_02063_b200 import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def gp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2312_02063_b200 import binding
    binding.lib()          # must load: no fallback
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def stream_and_assemble(gp, w, periods, nbins, want, slab_bytes, t0=None):
    """Consumer: copies every chunk into its place of a full-size tensor and adds a checksum,
    all on the consumer stream."""
    nc, npd = w.ncurves, len(periods)
    full = {k: torch.full((nc, npd, nbins), -77, dtype=torch.int32 if k == "count" else torch.float32,
                          device="cuda") for k in want}
    seen, checks = [], []
    cstream = torch.cuda.Stream()

    def consumer(ch):
        assert torch.cuda.current_stream() == cstream
        seen.append((ch["curve0"], ch["ncurves"], ch["period0"], ch["nperiods"], ch["slot"]))
        c0, c1 = ch["curve0"], ch["curve0"] + ch["ncurves"]
        p0, p1 = ch["period0"], ch["period0"] + ch["nperiods"]
        for k in want:
            full[k][c0:c1, p0:p1].copy_(ch[k])
        checks.append(ch[want[-1]].double().sum())

    gp.gpfc_fold_stream(dev(w.times), dev(w.flux), dev(w.offsets), dev(periods), nbins, consumer,
                        t0=None if t0 is None else dev(t0), want=want, slab_bytes=slab_bytes,
                        consumer_stream=cstream)
    torch.cuda.synchronize()
    return full, seen, [float(c) for c in checks]


def test_stream_chunks_of_curves_match_monolithic(gp, ref):
    w = workloads.config4(ncurves=23, nperiods=300)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    nb = w.nbins
    s, c, nrm = gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), dev(periods), nb)
    torch.cuda.synchronize()
    row = 300 * nb * 4 * 3
    full, seen, checks = stream_and_assemble(gp, w, periods, nb, ("sum", "count", "norm"), 4 * row + 100)
    assert [x[1] for x in seen] == [4, 4, 4, 4, 4, 3] and [x[0] for x in seen] == [0, 4, 8, 12, 16, 20]
    assert all(x[2] == 0 and x[3] == 300 for x in seen)
    assert [x[4] for x in seen] == [0, 1, 0, 1, 0, 1]
    assert torch.equal(full["sum"], s) and torch.equal(full["count"], c) and torch.equal(full["norm"], nrm)
    tot = sum(checks)
    assert abs(tot - float(nrm.double().sum())) <= 1e-6 * max(1.0, abs(tot))
    # norm only: a third of the slab per curve, so three times the curves per chunk
    full, seen, _ = stream_and_assemble(gp, w, periods, nb, ("norm",), 4 * row + 100)
    assert [x[1] for x in seen] == [12, 11]
    assert torch.equal(full["norm"], nrm)


def test_stream_chunks_of_periods_within_a_curve(gp, ref):
    """One curve's profiles larger than the slab: the chunks are runs of periods."""
    w = workloads.config1(nperiods=1000)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    for nb in (256, 1024):
        s, c, nrm = gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), dev(periods), nb)
        torch.cuda.synchronize()
        full, seen, _ = stream_and_assemble(gp, w, periods, nb, ("sum", "count", "norm"), 130 * nb * 12)
        assert [x[3] for x in seen] == [130] * 7 + [90] and all(x[0] == 0 and x[1] == 1 for x in seen)
        assert torch.equal(full["sum"], s) and torch.equal(full["count"], c) and torch.equal(full["norm"], nrm)


def test_stream_ragged_batch_t0_and_default_slab(gp, ref):
    w = workloads.ragged_batch(nperiods=40)
    periods = ref.make_period_grid(0.3, 7.0, w.nperiods, workloads.GRID_UNIFORM_PERIOD)
    t0 = np.linspace(-1.0, 2.0, w.ncurves)
    s, c, nrm = gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), dev(periods), 64, t0=dev(t0))
    torch.cuda.synchronize()
    full, seen, _ = stream_and_assemble(gp, w, periods, 64, ("count", "norm"), 0, t0=t0)
    assert len(seen) == 1 and seen[0][1] == w.ncurves
    assert torch.equal(full["count"], c) and torch.equal(full["norm"], nrm)
    full, seen, _ = stream_and_assemble(gp, w, periods, 64, ("norm",), 40 * 64 * 4, t0=t0)
    assert len(seen) == w.ncurves
    assert torch.equal(full["norm"], nrm)


def test_stream_consumer_error_and_arguments(gp, ref):
    w = workloads.config0()
    periods = ref.make_period_grid(w.pmin, w.pmax, 50, w.grid_mode)
    args = (dev(w.times), dev(w.flux), dev(w.offsets), dev(periods), 64)

    def bad(ch):
        raise RuntimeError("consumer failed")

    with pytest.raises(RuntimeError, match="consumer failed"):
        gp.gpfc_fold_stream(*args, bad)
    torch.cuda.synchronize()
    with pytest.raises(gp.GpfcError):
        gp.gpfc_fold_stream(*args, lambda ch: None, want=())
    # the library still works afterwards
    got = []
    gp.gpfc_fold_stream(*args, lambda ch: got.append(ch["norm"].clone()))
    torch.cuda.synchronize()
    assert torch.equal(got[0], gp.gpfc_fold_batch(*args)[2])


def test_host_path_norm_only_and_period_chunks(gp, ref):
    """gpfc_fold_batch_host runs on gpfc_fold_stream: norm-only output and a curve whose
    profiles exceed the 512 MB slab (config 3's shape, reduced) come back complete."""
    w = workloads.config1(nperiods=600)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    s, c, nrm = gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), dev(periods), 256)
    torch.cuda.synchronize()
    hn = np.full((1, 600, 256), -5, np.float32)
    gp.gpfc_fold_batch_host(w.times, w.flux, w.offsets, periods, 256, out_norm=hn)
    assert np.array_equal(hn, nrm.cpu().numpy())
    w3 = workloads.config3(nperiods=150000)      # 150,000 x 1,024 x 12 B = 1.84 GB: two period chunks
    p3 = ref.make_period_grid(w3.pmin, w3.pmax, w3.nperiods, w3.grid_mode)
    s, c, nrm = gp.gpfc_fold_batch(dev(w3.times), dev(w3.flux), dev(w3.offsets), dev(p3), 1024)
    torch.cuda.synchronize()
    hs, hn = np.empty((1, 150000, 1024), np.float32), np.empty((1, 150000, 1024), np.float32)
    hc = np.empty((1, 150000, 1024), np.uint32)
    gp.gpfc_fold_batch_host(w3.times, w3.flux, w3.offsets, p3, 1024, out_sum=hs, out_count=hc, out_norm=hn)
    assert np.array_equal(hs, s.cpu().numpy()) and np.array_equal(hn, nrm.cpu().numpy())
    assert np.array_equal(hc.view(np.uint32), c.cpu().numpy().view(np.uint32))
