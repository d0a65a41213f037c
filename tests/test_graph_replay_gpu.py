"""Launch sequences replayed as CUDA graphs (mvd_api.cu: run_graphed) must never serve a stale capture: the same handle is
driven through changing plane counts, buffers, settings and entry points, and every result is compared bit for bit
with a fresh handle that never replays anything."""
import numpy as np
import pytest
import torch

from paper_1503_07998_b200 import binding, build, synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


def _fresh(views, psfs, T, **kw):
    return binding.deconvolve(views, psfs, T, 1e-6, path=binding.PATH_FFT, **kw)


def test_one_handle_many_calls():
    V, N, W, H, K, T = 2, 12, 64, 64, 9, 3          # launch-bound: every device-resident call qualifies for replay
    pr = synth.make_problem(V, N, W, H, K, T, seed=77, psf="random")
    other = synth.random_views(V, N, W, H, seed=78, lo=0, hi=3000)
    dv = torch.from_numpy(pr.views.view(np.int16)).cuda()
    dv2 = torch.from_numpy(other.view(np.int16)).cuda()
    st = torch.cuda.Stream()
    with binding.Mvd(W, H, V, pr.psfs, K, T, 1e-6, binding.PATH_FFT) as m:
        def run(buf, n, out=None):
            out = torch.empty((n, H, W), dtype=torch.float32, device="cuda") if out is None else out
            sub = buf.view(V, N, H, W)[:, :n].contiguous()
            m.deconvolve_planes(sub, out, n, st)
            st.synchronize()
            return out.cpu().numpy()

        ref12 = _fresh(pr.views, pr.psfs, T)
        a = run(dv, 12); b = run(dv, 12); c = run(dv, 12)                    # capture, replay, replay
        assert np.array_equal(a, ref12) and np.array_equal(b, ref12) and np.array_equal(c, ref12)
        assert np.array_equal(run(dv2, 12), _fresh(other, pr.psfs, T))       # other buffers, same shape
        assert np.array_equal(run(dv, 5), _fresh(pr.views[:, :5], pr.psfs, T))   # other plane count (odd)
        assert np.array_equal(run(dv, 12), ref12)                            # and back
        # the same INPUT tensor with new contents: a replay reads what is there now
        keep = dv.clone()
        out = torch.empty((12, H, W), dtype=torch.float32, device="cuda")
        run(keep, 12, out)
        keep.copy_(dv2)
        assert np.array_equal(run(keep, 12, out), _fresh(other, pr.psfs, T))
        # settings that change the launch sequence invalidate the captures
        m.set_chunk_planes(4)
        assert np.array_equal(run(dv, 12), ref12)
        m.set_chunk_planes(0)
        m.set_update_mode(binding.UPDATE_PRODUCT)
        prod = _fresh(pr.views, pr.psfs, T, product=True)
        assert np.array_equal(run(dv, 12), prod) and np.array_equal(run(dv, 12), prod)
        m.set_update_mode(binding.UPDATE_SEQUENTIAL)
        assert np.array_equal(run(dv, 12), ref12)
        # host pipeline between device-resident calls (shared slots, its own per-batch captures), twice
        hv = torch.from_numpy(pr.views.view(np.int16)).pin_memory()
        ho = torch.empty((N, H, W), dtype=torch.float32).pin_memory()
        for _ in range(2):
            m.deconvolve_planes(dv, torch.empty((12, H, W), dtype=torch.float32, device="cuda"), 12, st)   # not synchronised
            m.deconvolve_host(hv, ho, N)
            assert np.array_equal(ho.numpy(), ref12)
        m.set_batch_planes(4)
        m.deconvolve_host(hv, ho, N)
        assert np.array_equal(ho.numpy(), ref12)
        assert np.array_equal(run(dv, 12), ref12)


def test_forked_resident_calls_then_host_pipeline():
    """Config 2's shape: the device-resident call forks to the internal streams (and is replayed as a graph), the host
    pipeline follows without a synchronisation in between -- the combination that once raced on the slots' scratch."""
    cfg = synth.config(2).with_planes(256)
    psfs = synth.config_psfs(2)
    base = synth.views(cfg, range(4), psfs)
    views = np.ascontiguousarray(np.tile(base, (1, 64, 1, 1)))
    dv = torch.from_numpy(views.view(np.int16)).cuda()
    hv = torch.from_numpy(views.view(np.int16)).pin_memory()
    ho = torch.empty((cfg.N, cfg.H, cfg.W), dtype=torch.float32).pin_memory()
    do = torch.empty((cfg.N, cfg.H, cfg.W), dtype=torch.float32, device="cuda")
    st = torch.cuda.Stream()
    with binding.Mvd(cfg.W, cfg.H, cfg.V, psfs, cfg.K, cfg.T, cfg.eps, binding.PATH_FFT) as m:
        m.reserve(cfg.N)
        for _ in range(3):
            m.deconvolve_planes(dv, do, cfg.N, st)
        m.deconvolve_host(hv, ho, cfg.N)
        st.synchronize()
        assert torch.equal(ho, do.cpu())
        m.deconvolve_planes(dv, do, cfg.N, st)
        m.deconvolve_host(hv, ho, cfg.N)
        st.synchronize()
        assert torch.equal(ho, do.cpu())
    # all 64 copies of the four base planes agree (planes are independent; pairs repeat every four planes)
    assert torch.equal(do[:4].cpu().repeat(64, 1, 1), do.cpu())
