"""spegg_offsets_static -- the one entry point of libspegg that allocates nothing -- against the scan of
the ordinary step.

Why the entry point exists: a caller that cannot allocate device memory where it stands (a plug-in inside
an application whose allocator owns the GPU, a callback under an allocator lock, a loop that cannot take
cudaMalloc's device-wide synchronisation) has no workspace to give to spegg_create.  For it the library
carries the scan's scratch as a fixed ~34 KB array in its own image; the limit is
SPEGG_STATIC_MAX_N = 4,194,304 adults per call and one call at a time per GPU.

What is checked: on the fecundities f[] that real steps of config 2 drew (read back through the debug
view), the new call returns exactly the offsets off[] and the neonate count M_t that the step's own scan
(k_fec_scan, scratch in the caller's workspace) produced -- integers, so the bar is equality, as in
tests/test_gpu_parity.py.  It is called twice in a row on different inputs, the second shorter than the
first, so leftovers of the first call in the shared array (aggregates, group counters, ticket) would
show.  This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It passes alone in a fresh process (the first call then also performs the
one-time address look-up) and after the rest of the suite."""
import os
import re

import numpy as np
import pytest

from paper_1603_09255_b200 import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_static_entry_point_source_makes_no_allocation():
    """No GPU needed: the file that holds the entry point calls no allocating CUDA routine (comments aside)
    and resolves its scratch array through cudaGetSymbolAddress before any kernel sees it."""
    src = open(os.path.join(ROOT, "paper_1603_09255_b200", "csrc", "spegg_static.cu")).read()
    code = re.sub(r"//[^\n]*|/\*.*?\*/", "", src, flags=re.S)
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemPool", "new ", "malloc(", "std::vector"):
        assert banned not in code, banned
    assert "static __device__ __align__(256)" in code
    assert "cudaGetSymbolAddress(&p, g_static_scratch)" in code
    # the array's name appears in host code only as the argument of that look-up
    host = code[code.index("int static_scratch"):]
    assert host.count("g_static_scratch") == 1


@pytest.fixture(scope="module")
def binding():
    from paper_1603_09255_b200 import binding as b
    from paper_1603_09255_b200 import build
    build.build()
    b.load()
    return b


def _step_fecundities(binding, scale, steps, seed=1):
    """f[], off[], M_t of `steps` consecutive debug steps of config 2 (the existing path)."""
    import parity
    cfg = workloads.config(2, scale=scale, seed=seed)
    sim = binding.Sim(cfg, debug=True)
    parity.load_initial(sim, cfg)
    out = []
    for _ in range(steps):
        sim.step(1)
        d = sim.read_debug(0)
        assert sim.status() == 0          # no overflow: m_t is the untruncated sum
        out.append((d["f"].copy(), d["off"].copy(), d["m_t"]))
    sim.close()
    return out


@pytest.mark.gpu
def test_offsets_static_matches_the_step_scan_twice_in_a_row(binding):
    import torch
    # step 1 starts from N0 adults, step 2 from fewer survivors: the second input is shorter, so tile
    # aggregates and the ticket the first call left behind lie inside the range the second must clear
    (f1, off1, m1), (f2, off2, m2) = _step_fecundities(binding, scale=0.4, steps=2)
    assert len(f1) > 8 * 1024 and len(f1) % 1024 != 0 and len(f2) != len(f1)   # several tiles and a ragged tail
    dev = torch.device("cuda:0")
    n_max = max(len(f1), len(f2))
    # every buffer exists BEFORE the calls; the calls themselves create nothing
    d_f = torch.zeros(n_max, dtype=torch.uint8, device=dev)
    d_off = torch.zeros(n_max, dtype=torch.int32, device=dev)
    d_tot = torch.zeros(2, dtype=torch.int64, device=dev)
    d_off2 = torch.zeros(n_max, dtype=torch.int32, device=dev)
    d_f2 = torch.from_numpy(f2).to(dev)
    d_f[:len(f1)] = torch.from_numpy(f1).to(dev)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(dev)
    binding.offsets_static(d_f, d_off, d_tot[0:1], n=len(f1))
    binding.offsets_static(d_f2, d_off2, d_tot[1:2], n=len(f2))      # same stream: ordered, no overlap
    torch.cuda.synchronize()
    got1 = d_off[:len(f1)].cpu().numpy().view(np.uint32)
    got2 = d_off2[:len(f2)].cpu().numpy().view(np.uint32)
    tot = d_tot.cpu().numpy()
    assert np.array_equal(got1, off1) and int(tot[0]) == m1 == int(f1.sum(dtype=np.int64))
    assert np.array_equal(got2, off2) and int(tot[1]) == m2 == int(f2.sum(dtype=np.int64))
    # ... and back to the first input: a third call after a shorter one
    d_off.zero_()
    binding.offsets_static(d_f, d_off, d_tot[0:1], n=len(f1))
    torch.cuda.synchronize()
    assert np.array_equal(d_off[:len(f1)].cpu().numpy().view(np.uint32), off1)
    free_mid, _ = torch.cuda.mem_get_info(dev)
    binding.offsets_static(d_f, d_off, d_tot[0:1], n=len(f1))
    binding.offsets_static(d_f2, d_off2, d_tot[1:2], n=len(f2))
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info(dev)
    assert free_after == free_mid, "device memory in use changed across two calls of the no-allocation entry point"
    assert free_before >= free_mid     # (the very first call may load the kernel's module; it never frees)


@pytest.mark.gpu
def test_offsets_static_limit_and_edges(binding):
    import torch
    dev = torch.device("cuda:0")
    g = torch.Generator(device="cpu").manual_seed(7)
    n = binding.STATIC_MAX_N
    f = torch.randint(0, 17, (n + 1,), dtype=torch.uint8, generator=g)    # lambda <= 2: fecundities stay small
    d_f = f.to(dev)
    d_off = torch.zeros(n + 1, dtype=torch.int32, device=dev)
    d_tot = torch.full((1,), -1, dtype=torch.int64, device=dev)
    # one adult too many: refused with the limit's own error code, nothing launched, outputs untouched
    with pytest.raises(binding.SpeggError) as e:
        binding.offsets_static(d_f, d_off, d_tot, n=n + 1)
    assert e.value.code == binding.ELIMIT and "maximum" in str(e.value)
    torch.cuda.synchronize()
    assert int(d_tot.item()) == -1 and int(d_off.abs().sum().item()) == 0
    # exactly the maximum: all 4,096 tiles and 128 complete groups of the array in use
    binding.offsets_static(d_f, d_off, d_tot, n=n)
    ref = np.cumsum(f.numpy()[:n].astype(np.int64))
    assert np.array_equal(d_off[:n].cpu().numpy().view(np.uint32), (ref - f.numpy()[:n]).astype(np.uint32))
    assert int(d_tot.item()) == int(ref[-1])
    # right after the largest call: tiny, empty, tile-aligned and byte-misaligned inputs
    for lo, cnt in ((0, 1), (0, 0), (0, 1024), (0, 2048), (1, 1023), (3, 4099), (2, 31)):
        d_tot.fill_(-1)
        d_off.zero_()
        binding.offsets_static(d_f[lo:lo + cnt], d_off[:max(cnt, 1)], d_tot, n=cnt)
        h = f.numpy()[lo:lo + cnt].astype(np.int64)
        assert int(d_tot.item()) == int(h.sum()), (lo, cnt)
        assert np.array_equal(d_off[:cnt].cpu().numpy().astype(np.int64), np.cumsum(h) - h), (lo, cnt)
    # NULL outputs are a parameter error, not a fault
    assert binding.load().spegg_offsets_static(d_f.data_ptr(), 10, None, d_tot.data_ptr(), None) == binding.EINVAL
    assert binding.load().spegg_offsets_static(d_f.data_ptr(), 10, d_off.data_ptr(), None, None) == binding.EINVAL
