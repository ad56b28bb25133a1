"""-m gpu: what include/saltband.h promises about the boundary itself.

* concurrent compute calls from two host threads on two streams with the same handles give results
  bit-identical to serial calls (per-stream workspaces owned by the bands handle);
* sb_chi2 and sb_bandflux_grad only enqueue work: a warmed-up call can be captured into a CUDA graph and
  the replay gives the same outputs (no allocation, no host synchronisation inside the call);
* a pack (sb_pack_observations) changes nothing but the work done per call: bit-identical outputs,
  fewer launches; a pack that does not belong to the batch is refused;
* misaligned gradient outputs are refused (they are written as 16-byte vectors)."""
import threading

import numpy as np
import pytest

import oracle
import sbgpu
import workloads

pytestmark = pytest.mark.gpu


def _prepare(config, **kw):
    wl = workloads.make_workload(config, **kw)
    true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()})["flux"]
    workloads.attach_data(wl, true)
    return wl


def _device_args(wl, dev):
    import torch

    import paper_2504_08081_b200 as sb

    f = lambda a: torch.as_tensor(np.asarray(a, dtype=np.float32)).to(dev)  # noqa: E731
    i = lambda a: torch.as_tensor(np.asarray(a, dtype=np.int32)).to(dev)  # noqa: E731
    return dict(dtype=sb.SB_F32, n_sn=wl.n_sn, n_samples=wl.n_samples, n_obs_total=wl.n_obs_total,
                obs_offset=i(wl.obs_offset), time=f(wl.time), band=i(wl.band), zp=f(wl.zp), z=f(wl.z),
                x0=f(wl.theta["x0"]), x1=f(wl.theta["x1"]), c=f(wl.theta["c"]), t0=f(wl.theta["t0"])), f(wl.flux), f(wl.fluxerr)


def test_two_threads_two_streams_equal_serial_calls(cuda_device):
    import torch

    import paper_2504_08081_b200 as sb

    wls = [_prepare(2, n_sn=700), _prepare(2, n_sn=900, seed_offset=3)]
    model, bands = sbgpu.load_handles(wls[0])
    args = [_device_args(w, cuda_device) for w in wls]
    serial = []
    for w, (kw, fl, fe) in zip(wls, args):
        chi = torch.empty(w.n_sn, dtype=torch.float32, device=cuda_device)
        flux = torch.empty(w.n_evals, dtype=torch.float32, device=cuda_device)
        sb.sb_chi2(model, bands, flux=fl, fluxerr=fe, out_chi2=chi, out_flux=flux, **kw)
        torch.cuda.synchronize()
        serial.append((chi.cpu().numpy().copy(), flux.cpu().numpy().copy()))
    results = [None, None]
    errors = []

    def worker(k):
        try:
            w, (kw, fl, fe) = wls[k], args[k]
            stream = torch.cuda.Stream(device=cuda_device)
            chi = torch.empty(w.n_sn, dtype=torch.float32, device=cuda_device)
            flux = torch.empty(w.n_evals, dtype=torch.float32, device=cuda_device)
            with torch.cuda.stream(stream):
                for _ in range(20):  # many overlapping calls on both streams
                    sb.sb_chi2(model, bands, flux=fl, fluxerr=fe, out_chi2=chi, out_flux=flux, **kw)
            stream.synchronize()
            results[k] = (chi.cpu().numpy(), flux.cpu().numpy())
        except Exception as exc:  # pragma: no cover
            errors.append(exc)

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for k in range(2):
        assert np.array_equal(results[k][0], serial[k][0]) and np.array_equal(results[k][1], serial[k][1])


@pytest.mark.parametrize("mode", ["chi2", "grad"])
@pytest.mark.parametrize("use_pack", [False, True])
def test_calls_can_be_captured_into_a_cuda_graph(cuda_device, mode, use_pack):
    import torch

    import paper_2504_08081_b200 as sb

    wl = _prepare(4, n_sn=300)
    model, bands = sbgpu.load_handles(wl)
    kw, fl, fe = _device_args(wl, cuda_device)
    n_ev, n_u = wl.n_evals, wl.n_sn
    chi = torch.zeros(n_u, dtype=torch.float32, device=cuda_device)
    flux = torch.zeros(n_ev, dtype=torch.float32, device=cuda_device)
    dflux = torch.zeros(n_ev * 4, dtype=torch.float32, device=cuda_device)
    dchi = torch.zeros(n_u * 4, dtype=torch.float32, device=cuda_device)
    stream = torch.cuda.Stream(device=cuda_device)
    with torch.cuda.stream(stream):
        if use_pack:
            kw["pack"] = sb.sb_pack_observations(model, bands, dtype=sb.SB_F32, n_sn=wl.n_sn, z=kw["z"])

        def call():
            if mode == "chi2":
                sb.sb_chi2(model, bands, flux=fl, fluxerr=fe, out_chi2=chi, out_flux=flux, **kw)
            else:
                sb.sb_bandflux_grad(model, bands, flux=fl, fluxerr=fe, out_flux=flux, out_dflux=dflux, out_chi2=chi,
                                    out_dchi2=dchi, **kw)

        call()  # warm-up: the first call on a stream may allocate the stream's workspace
        stream.synchronize()
        want = [t.clone() for t in (chi, flux, dflux, dchi)]
        for t in (chi, flux, dflux, dchi):
            t.zero_()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            call()  # only enqueues: any allocation or synchronisation here would fail the capture
        for t in (chi, flux, dflux, dchi):
            t.zero_()
        graph.replay()
        stream.synchronize()
    for a, b in zip(want, (chi, flux, dflux, dchi)):
        assert torch.equal(a, b)


def test_pack_is_bit_identical_and_saves_the_sort(cuda_device):
    import paper_2504_08081_b200 as sb

    wl = _prepare(5, n_sn=9000)  # > 8192 supernovae: the two-kernel z-order sort
    handles = sbgpu.load_handles(wl)
    for mode in ("chi2", "grad"):
        a = sbgpu.run_gpu(wl, mode=mode, handles=handles)
        b = sbgpu.run_gpu(wl, mode=mode, handles=handles, use_pack=True)
        assert a["form"] == b["form"] == "tiled"
        assert a["launches"] == 3 and b["launches"] == 1  # z-hist + z-scatter + main  vs  main only
        for key in ("flux", "chi2") + (("dflux", "dchi2") if mode == "grad" else ()):
            assert np.array_equal(a[key], b[key]), (mode, key)
    # a pack built for another batch is refused
    import torch

    other = sb.sb_pack_observations(handles[0], handles[1], dtype=sb.SB_F32, n_sn=10,
                                    z=torch.zeros(10, dtype=torch.float32, device=cuda_device))
    kw, fl, fe = _device_args(wl, cuda_device)
    chi = torch.empty(wl.n_sn, dtype=torch.float32, device=cuda_device)
    with pytest.raises(sb.SaltbandError, match="invalid argument"):
        sb.sb_chi2(*handles, flux=fl, fluxerr=fe, out_chi2=chi, pack=other, **kw)


def test_misaligned_gradient_outputs_are_refused(cuda_device):
    import ctypes as C

    import torch

    import paper_2504_08081_b200 as sb
    from paper_2504_08081_b200 import api

    wl = _prepare(2, n_sn=64)
    model, bands = sbgpu.load_handles(wl)
    kw, fl, fe = _device_args(wl, cuda_device)
    buf = torch.empty(wl.n_evals * 4 + 4, dtype=torch.float32, device=cuda_device)
    bt = api._batch(kw["dtype"], wl.n_sn, 1, kw["obs_offset"], kw["time"], kw["band"], kw["zp"], kw["z"], kw["x0"],
                    kw["x1"], kw["c"], kw["t0"], wl.n_obs_total)
    rc = api._load().sb_bandflux_grad(model._h, bands._h, C.byref(bt), None, None, None, buf.data_ptr() + 4, None, None,
                                      torch.cuda.current_stream().cuda_stream)
    assert rc == -1  # SB_EINVAL
    rc = api._load().sb_bandflux_grad(model._h, bands._h, C.byref(bt), None, None, None, buf.data_ptr(), None, None,
                                      torch.cuda.current_stream().cuda_stream)
    assert rc == 0
    torch.cuda.synchronize()
