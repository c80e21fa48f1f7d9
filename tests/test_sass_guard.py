"""The payload of the B200 path must keep moving through the async copy engine, not through registers.

`cuobjdump -sass` of the built library, read per kernel (no GPU needed): every contiguous form of kv_move_shot_plain,
kv_move_shot and kv_move_bulk holds a bulk load global -> shared (UBLKCP.S.G, PTX cp.async.bulk ... shared::cluster.global)
and a bulk store shared -> global (UBLKCP.G.S); every HND form also holds the tensor copies that do the [head][token]
transposition (UTMALDG / UTMASTG, PTX cp.async.bulk.tensor).  The plain kernel moves payload with nothing else: it has
no LDG / STG wider than a table read.  A refactor that quietly puts the payload back into registers fails here.
(The histogram of profiles/r02_sass_opcodes.md, as an assertion.)"""
import re
import shutil
import subprocess

import pytest

from paper_2606_31093_b200 import kvtier as kv


@pytest.fixture(scope="module")
def sass():
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    try:
        out = subprocess.run([exe, "-sass", kv.LIB_PATH], check=True, capture_output=True, text=True).stdout
    except (OSError, subprocess.CalledProcessError) as e:  # no CUDA toolkit on this machine
        pytest.skip(f"cuobjdump unavailable: {e}")
    funcs = {}
    name = None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            funcs[name] = []
        elif name is not None:
            m = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
            if m:
                funcs[name].append(m.group(1))
    assert funcs, "no SASS functions found"
    return funcs


def forms(sass, kernel):
    """{(N, trans): opcodes} of kvt::<kernel><N, trans> from the mangled names (..IL i<N> EL b<0|1> E..)."""
    out = {}
    for name, ops in sass.items():
        m = re.search(rf"3kvt\d+{kernel}ILi(\d+)ELb([01])EEEv", name)
        if m:
            out[(int(m.group(1)), m.group(2) == "1")] = ops
    return out


@pytest.mark.parametrize("kernel", ["kv_move_shot_plain", "kv_move_shot", "kv_move_bulk"])
def test_async_copy_kernels_move_payload_with_bulk_and_tensor_copies(sass, kernel):
    f = forms(sass, kernel)
    assert len(f) == 6, f"{kernel}: expected 3 table sizes x (contiguous, HND), found {sorted(f)}"
    assert {n for n, _ in f} >= {0}, "the tables-in-device-memory form is missing"
    for (n, trans), ops in f.items():
        has = lambda prefix: any(o.startswith(prefix) for o in ops)  # noqa: E731
        assert has("UBLKCP.S.G"), f"{kernel}<{n},{trans}>: no bulk load global -> shared"
        assert has("UBLKCP.G.S"), f"{kernel}<{n},{trans}>: no bulk store shared -> global"
        if trans:
            assert has("UTMALDG"), f"{kernel}<{n},{trans}>: no tensor load (the copy engine's transposition)"
            assert has("UTMASTG"), f"{kernel}<{n},{trans}>: no tensor store"
        else:
            assert not has("UTMALDG") and not has("UTMASTG"), f"{kernel}<{n},{trans}>: tensor copies in a contiguous form"
        assert any(o.startswith("SYNCS") for o in ops), f"{kernel}<{n},{trans}>: no mbarrier"


def test_plain_kernel_touches_payload_with_nothing_else(sass):
    for (n, trans), ops in forms(sass, "kv_move_shot_plain").items():
        wide = [o for o in ops if re.match(r"(LDG|STG|LDS|STS)\b.*\.(64|128)", o) and ".CONSTANT" not in o]
        stores = [o for o in ops if o.startswith(("STG", "STS", "LDS"))]
        assert not stores, f"kv_move_shot_plain<{n},{trans}> stores or reads shared memory with lane instructions: {stores}"
        assert not wide, f"kv_move_shot_plain<{n},{trans}> has wide lane loads: {wide}"
        assert len(ops) <= 320, f"kv_move_shot_plain<{n},{trans}> grew to {len(ops)} instructions (the short kernel of the small calls)"


def test_no_tensor_core_instructions_anywhere(sass):
    """A permutation copy is not a contraction (BASELINE.json:north_star item 2)."""
    for name, ops in sass.items():
        bad = [o for o in ops if o.startswith(("HMMA", "IMMA", "UTCHMMA", "UTCIMMA", "UTCQMMA", "QMMA", "BMMA", "DMMA"))]
        assert not bad, f"{name}: {bad[:3]}"
