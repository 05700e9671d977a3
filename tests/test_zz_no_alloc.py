"""GPU test of fizzy_count_nonfinite_static (include/fizzy.h), the one entry point of libfizzy.so that needs no context,
no workspace and no allocation: its scratch is an array built into the library.  It exists for callers that are handed
device pointers to the fields and may not allocate -- a monitoring / output hook running inside a solver whose pool
allocator owns the whole GPU, where a cudaMalloc would fail or stall the solver's streams (it synchronises the device).

What is checked: the count equals the one the existing path (fizzy_check_finite on a context holding the same fields)
returns -- integer work, so the bar is equality, as in test_check_finite -- on two calls in a row with different
contents (the built-in array keeps the previous call's data, so a stale partial count would show up in the second call);
ragged sizes around the 4096-value chunk against a plain torch count; the size limit and the other rejections; and that
device memory in use does not change across a call.

The file sorts last on purpose (pytest -x stops at the first failure and this entry point lies outside the hot path) and
passes alone in a fresh process as well as after the other GPU tests: it depends on no state they leave behind."""
import numpy as np
import pytest

from paper_2502_04189_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fz():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2502_04189_b200 import binding
    return binding


def _device_fields(g, torch):
    """The context's fields as device tensors (fizzy_get_fields with device pointers)."""
    names = ["u", "v", "w", "p", "phi"] + (["T"] if g.heat else [])
    out = {k: torch.empty(g.shape, dtype=torch.float64, device=g.device) for k in names}
    g.fizzy_get_fields(**out)
    g.stream.synchronize()
    return [out[k] for k in names]


def test_matches_fizzy_check_finite_on_two_calls_in_a_row(fz):
    import torch
    # config 5's physics (six fields, walls, stretched z) on a grid of 24.5 chunks: the last block is half empty
    cfg, f, dt, _ = W.make(4, grid=(64, 32, 49), ndrops=2, radius=0.3)
    g = fz.Fizzy(cfg)
    # first call: seven bad values, among them the very first and the very last value of a field
    bad = {k: a.copy() for k, a in f.items()}
    bad["u"][0, 0, 0] = np.inf
    bad["u"][48, 31, 63] = np.nan
    bad["v"][17, 5, 40] = -np.inf
    bad["p"][48, 31, 62] = np.nan
    bad["phi"][20, 20, 20] = np.nan
    bad["T"][3, 4, 5] = np.nan
    bad["T"][48, 0, 0] = np.inf
    g.set_fields_numpy(**bad)
    expect1 = g.fizzy_check_finite()
    assert expect1 == 7
    got1 = fz.fizzy_count_nonfinite_static(_device_fields(g, torch), stream=g.stream)
    assert got1 == expect1
    # second call, right after: fewer bad values in other places (a count left over from the first call would be seen)
    bad = {k: a.copy() for k, a in f.items()}
    bad["w"][10, 10, 10] = np.nan
    bad["phi"][48, 31, 63] = np.inf
    g.set_fields_numpy(**bad)
    expect2 = g.fizzy_check_finite()
    assert expect2 == 2
    got2 = fz.fizzy_count_nonfinite_static(_device_fields(g, torch), stream=g.stream)
    assert got2 == expect2
    # and a healthy state after one RK3 step
    g.set_fields_numpy(**f)
    g.step(dt)
    assert g.fizzy_check_finite() == 0
    assert fz.fizzy_count_nonfinite_static(_device_fields(g, torch), stream=g.stream) == 0
    g.close()


@pytest.mark.parametrize("n", [1, 255, 4095, 4096, 4097, 3 * 4096 + 17, 1_000_003, 37])
def test_ragged_sizes_against_a_plain_count(fz, n):
    """Sizes around the chunk boundary, large then small (n = 37 after 1 000 003: 244 stale slots stay in the array)."""
    import torch
    gen = torch.Generator(device="cuda").manual_seed(1234 + n)
    fields = [torch.randn(n, dtype=torch.float64, device="cuda", generator=gen) for _ in range(3)]
    k = min(n, 11)
    for q, a in enumerate(fields):
        idx = torch.randperm(n, device="cuda", generator=gen)[:k]
        a[idx[: k // 2 + 1]] = float("nan")
        a[idx[k // 2 + 1:]] = float("inf") if q % 2 else float("-inf")
        a[n - 1] = float("nan")
    expect = int(sum((~torch.isfinite(a)).sum().item() for a in fields))
    torch.cuda.synchronize()
    assert fz.fizzy_count_nonfinite_static(fields) == expect
    assert fz.fizzy_count_nonfinite_static(fields[:1]) == int((~torch.isfinite(fields[0])).sum().item())
    # denormals, huge finite values and zeros are finite
    ok = torch.tensor([0.0, -0.0, 5e-324, 1.7976931348623157e308, -1.7976931348623157e308], dtype=torch.float64, device="cuda")
    assert fz.fizzy_count_nonfinite_static([ok]) == 0


def test_limits_and_rejections(fz):
    import torch
    a = torch.zeros(4096, dtype=torch.float64, device="cuda")
    assert fz.fizzy_count_nonfinite_static([a], n=0) == 0
    with pytest.raises(fz.FizzyError) as e:      # one value too many for the built-in array: refused, nothing is read
        fz.fizzy_count_nonfinite_static([a], n=fz.FIZZY_STATIC_MAX_VALUES + 1)
    assert e.value.status == fz.FIZZY_EINVAL and "FIZZY_STATIC_MAX_VALUES" in str(e.value)
    with pytest.raises(fz.FizzyError) as e:
        fz.fizzy_count_nonfinite_static([a] * (fz.FIZZY_STATIC_MAX_FIELDS + 1))
    assert e.value.status == fz.FIZZY_EINVAL
    with pytest.raises(fz.FizzyError) as e:
        fz.fizzy_count_nonfinite_static([], n=8)
    assert e.value.status == fz.FIZZY_EINVAL
    with pytest.raises(fz.FizzyError) as e:
        fz.fizzy_count_nonfinite_static([a], n=-1)
    assert e.value.status == fz.FIZZY_EINVAL
    with pytest.raises(fz.FizzyError) as e:      # pageable host memory: cannot be staged without allocating
        fz.fizzy_count_nonfinite_static([np.zeros(16)], n=16)
    assert e.value.status == fz.FIZZY_EINVAL and "device" in str(e.value)
    with pytest.raises(fz.FizzyError) as e:
        fz.fizzy_count_nonfinite_static([a, 0], n=16)
    assert e.value.status == fz.FIZZY_EINVAL
    assert fz.fizzy_count_nonfinite_static([a]) == 0   # still usable after the refusals


def test_largest_size_and_no_change_in_device_memory(fz):
    """n = FIZZY_STATIC_MAX_VALUES (one field of a 512^3 grid, every slot of the array in use), twice; the amount of free
    device memory is the same before and after the calls (the set-up of the first call in this process is excluded)."""
    import torch
    n = fz.FIZZY_STATIC_MAX_VALUES
    a = torch.zeros(n, dtype=torch.float64, device="cuda")
    a[n - 1] = float("nan")
    a[0] = float("inf")
    a[n // 2 + 4095] = float("nan")
    fz.fizzy_count_nonfinite_static([a[:16]])          # set-up call (loads the kernel on this device if nothing did yet)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    assert fz.fizzy_count_nonfinite_static([a]) == 3
    a[n - 1:].zero_()                                  # in place: no torch allocation between the two readings
    assert fz.fizzy_count_nonfinite_static([a]) == 2
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
