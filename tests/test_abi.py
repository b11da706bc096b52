"""The C-ABI library loads and exports every function include/pixclus.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

import paper_2104_06573_b200 as pix
from paper_2104_06573_b200 import build as pixbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "pixclus.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pix_[a-z_]+)\s*\(", text)))


def test_header_declares_the_boundary():
    names = declared_functions()
    for n in ("pix_create", "pix_clone", "pix_destroy", "pix_process", "pix_process_batch", "pix_process_batch_host",
              "pix_last_error"):
        assert n in names


def test_library_exports_every_declared_symbol():
    lib = ctypes.CDLL(pixbuild.build())
    for n in declared_functions():
        assert hasattr(lib, n), f"libpixclus.so does not export {n}"


def test_binding_names_match_header():
    assert set(pix.EXPORTS) == set(declared_functions())


def test_struct_layouts_match_header():
    """pix_params field order in the binding follows the header (argument marshalling only)."""
    text = open(os.path.join(ROOT, "include", "pixclus.h")).read()
    body = re.search(r"typedef struct \{([^}]*)\} pix_params;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = [f for decl in body.split(";") for f in re.findall(r"(\w+)\s*(?:,|$)", decl.strip().split(" ", 1)[-1]) if decl.strip()]
    assert [n for n, _ in pix.Params._fields_] == fields


def test_product_path_does_not_import_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2104_06573_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "oracle/" not in src.replace("shared with oracle/", ""), f
