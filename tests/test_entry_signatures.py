"""Host-side check (no GPU): every call that `__graft_entry__.smoke()` and `bench.py` make into the binding binds to the
binding's current Python signature. The smoke test only runs on the GPU box, so a binding whose argument list changed
(e.g. legs_loss_workspace_bytes gaining P) would otherwise be noticed only there."""
import ast
import inspect
import os

from paper_2311_18482_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _calls(path, module_alias="legs"):
    tree = ast.parse(open(path).read())
    for node in ast.walk(tree):
        if isinstance(node, ast.Call) and isinstance(node.func, ast.Attribute) and isinstance(node.func.value, ast.Name) \
                and node.func.value.id == module_alias:
            yield node


def _check(path):
    n = 0
    for call in _calls(path):
        name = call.func.attr
        target = getattr(binding, name, None)
        assert target is not None, f"{os.path.basename(path)}:{call.lineno}: binding has no attribute {name}"
        if not (inspect.isfunction(target) or inspect.isclass(target)):
            continue
        if any(isinstance(a, ast.Starred) for a in call.args) or any(k.arg is None for k in call.keywords):
            continue
        sig = inspect.signature(target)
        try:
            sig.bind(*[None] * len(call.args), **{k.arg: None for k in call.keywords})
        except TypeError as e:
            raise AssertionError(f"{os.path.basename(path)}:{call.lineno}: legs.{name}(...) does not bind: {e}")
        n += 1
    return n


def test_smoke_calls_bind_to_the_binding():
    assert _check(os.path.join(ROOT, "__graft_entry__.py")) >= 10


def test_bench_calls_bind_to_the_binding():
    assert _check(os.path.join(ROOT, "bench.py")) >= 20
