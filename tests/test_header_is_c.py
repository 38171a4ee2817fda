"""include/optimus_b200.h is plain C (it compiles as C99 with gcc), and the ctypes mirrors of binding.py have the
struct layouts the C compiler gives the header's structs (sizeof + offsetof of every field)."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "optimus_b200.h")

STRUCTS = ["opt_linear_member", "opt_linear_options", "opt_linear2_member", "opt_ln_linear2_member", "opt_layernorm_member",
           "opt_layernorm_bwd_member", "opt_bias_grad_member", "opt_chunk", "opt_host_copy"]


def _header_structs():
    """{struct name: [field names]} parsed from the header's `typedef struct { ... } name;` blocks."""
    text = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    out = {}
    for body, name in re.findall(r"typedef\s+struct\s*\{(.*?)\}\s*(\w+)\s*;", text, flags=re.S):
        fields = []
        for decl in body.split(";"):
            decl = decl.strip()
            if not decl:
                continue
            # "const void* x", "int32_t M, N, K", "float p0, p1, p2", "int32_t reserved[5]", "opt_linear2_member chain"
            first, *rest = [d.strip() for d in decl.split(",")]
            fields.append(re.sub(r"\[.*\]", "", first.split()[-1].lstrip("*")))
            fields += [re.sub(r"\[.*\]", "", r.lstrip("*")) for r in rest]
        out[name] = fields
    return out


def test_header_compiles_as_c99():
    r = subprocess.run(["gcc", "-x", "c", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-fsyntax-only", HEADER],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_every_struct_of_the_header_is_mirrored():
    assert sorted(_header_structs()) == sorted(STRUCTS)


def test_struct_layouts_match_the_ctypes_mirrors(tmp_path):
    sys.path.insert(0, ROOT)
    from paper_2607_02945_b200 import binding
    parsed = _header_structs()
    lines = ['#include <stddef.h>', '#include <stdio.h>', '#include "optimus_b200.h"', "int main(void) {"]
    for s in STRUCTS:
        lines.append('  printf("%s . %%zu\\n", sizeof(%s));' % (s, s))
        for f in parsed[s]:
            lines.append('  printf("%s %s %%zu\\n", offsetof(%s, %s));' % (s, f, s, f))
    lines += ["  return 0;", "}"]
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)])
    got = {}
    for ln in subprocess.check_output([str(exe)], text=True).splitlines():
        s, f, v = ln.split()
        got[(s, f)] = int(v)
    for s in STRUCTS:
        mirror = getattr(binding, s)
        assert [n for n, *_ in mirror._fields_] == parsed[s], s          # same fields, same order
        assert C.sizeof(mirror) == got[(s, ".")], s
        for f in parsed[s]:
            assert getattr(mirror, f).offset == got[(s, f)], (s, f)


def test_a_c_program_drives_the_abi(tmp_path):
    """A 30-line C caller: links against the .so, validates on the host (no GPU needed): a NULL descriptor and a
    misaligned member come back as the documented error codes with a message, nothing is launched."""
    sys.path.insert(0, ROOT)
    from paper_2607_02945_b200 import build
    lib = build.build()
    src = tmp_path / "caller.c"
    src.write_text(r'''
#include <stdio.h>
#include <string.h>
#include "optimus_b200.h"
int main(void) {
  opt_plan* plan = (opt_plan*)1;
  if (opt_linear_plan_create(NULL, 1, OPT_BF16, 0, &plan) != OPT_ERR_INVALID_ARG || plan != NULL) return 1;
  if (strlen(opt_last_error()) == 0) return 2;
  opt_layernorm_member m;
  memset(&m, 0, sizeof m);
  m.x = (const void*)0x1000; m.y = (void*)0x2008; m.ldx = 64; m.ldy = 64; m.rows = 4; m.D = 64; m.eps = 1e-5f;
  if (opt_layernorm_plan_create(&m, 1, OPT_BF16, OPT_BF16, 0, &plan) != OPT_ERR_ALIGNMENT || plan != NULL) return 3;
  opt_chunk c;
  memset(&c, 0, sizeof c);
  c.src = (const void*)0x1000; c.dst = (void*)0x1010; c.lds = 64; c.ldd = 64; c.rows = 2; c.width = 64; c.op = OPT_PW_RELU;
  if (opt_pointwise_plan_create(&c, 1, OPT_BF16, 0, &plan) != OPT_ERR_ALIAS) return 4;
  if (opt_plan_launch(NULL, NULL) != OPT_ERR_INVALID_ARG) return 5;
  if (strncmp(opt_version(), "liboptimus_b200", 15) != 0) return 6;
  if (opt_launch_count() != 0) return 7;
  puts("ok");
  return 0;
}
''')
    exe = tmp_path / "caller"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src),
                           lib, "-Wl,-rpath," + os.path.dirname(lib)])
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 0 and r.stdout.strip() == "ok", (r.returncode, r.stdout, r.stderr)
