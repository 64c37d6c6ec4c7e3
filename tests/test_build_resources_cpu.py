"""Resource guard for the hot kernels (CPU-only: reads the cross-compiled sm_100a image with cuobjdump).

The FP64 kernels sit at register counts that decide how many CTAs an SM holds, and ptxas moves them on small
source changes elsewhere: adding one field to NufftParams once pushed k_spread_mma<11> from 96 to 116 registers
(5 -> 4 CTAs per SM, 3.29 -> 3.58 ms) and a table lookup made k_legendre_adjoint<5, 8> spill (4.2 -> 4.9 ms),
both with every parity test still green.  The bounds are the occupancy steps DESIGN.md section 9 relies on."""
import re
import shutil
import subprocess

import pytest


def resources():
    from paper_2406_14542_b200 import build
    lib = build.build()
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    try:
        out = subprocess.run([exe, "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    except (OSError, subprocess.CalledProcessError):
        pytest.skip("cuobjdump not available")
    res = {}
    for m in re.finditer(r"Function (\S+):\s*\n\s*REG:(\d+) STACK:(\d+) SHARED:(\d+)", out):
        res[m.group(1)] = tuple(int(m.group(i)) for i in (2, 3, 4))
    return res


def find(res, *parts):
    hits = [v for k, v in res.items() if all(p in k for p in parts)]
    assert len(hits) == 1, (parts, len(hits))
    return hits[0]


def test_hot_kernels_keep_their_occupancy_step():
    res = resources()
    assert len(res) > 50
    # (mangled-name fragments, max registers, threads per CTA, CTAs per SM that must still fit)
    cases = [
        (("k_legendre_synth", "ILi4ELb0E"), 32, 16),
        (("k_legendre_adjoint", "ILi5ELi8ELb0E"), 32, 16),
        (("k_legendre_synth", "ILi4ELb1E"), 32, 16),          # ring-list variants (rSHT front end)
        (("k_legendre_adjoint", "ILi5ELi8ELb1E"), 32, 16),
        (("k_interp_mma", "ILi11E"), 128, 6),
        (("k_spread_mma", "ILi11E"), 128, 5),
        (("k_interp_mma", "ILi9E"), 128, 6),
        (("k_spread_mma", "ILi9E"), 128, 5),
    ]
    for parts, threads, ctas in cases:
        reg, stack, shared = find(res, *parts)
        assert stack == 0, (parts, "spills: STACK", stack)
        alloc = -(-reg * 32 // 256) * 256 * (threads // 32)      # registers are allocated per warp in units of 256
        assert alloc * ctas <= 65536, (parts, reg, "registers: fewer than", ctas, "CTAs per SM")
        assert shared * ctas <= 233472, (parts, shared)


def test_theta_chain_fits_one_cta_per_sm():
    res = resources()
    for name in ("k_theta_chain_syn", "k_theta_chain_adj"):
        hits = [v for k, v in res.items() if name in k and "8192" in k and "7double2" in k]
        assert hits, name
        for reg, stack, shared in hits:
            assert reg <= 128, (name, reg)
