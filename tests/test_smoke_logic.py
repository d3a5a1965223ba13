"""The driver's smoke() (repo root, __graft_entry__.py) executed against the host emulation of the library: every
assertion it will make on the first contact with a B200 holds for the library's own kernels without a GPU."""
import __graft_entry__ as entry
from backends import BACKENDS


def test_smoke_assertions_hold_in_emulation(capsys):
    be = BACKENDS["simt"]
    with be.ctx():
        entry.smoke(be)
    assert "smoke ok" in capsys.readouterr().out
