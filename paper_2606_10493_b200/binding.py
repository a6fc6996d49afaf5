# placeholder, replaced below
class SlpMoeLayer: pass
class SlpError(Exception): pass
def lib(): raise RuntimeError
def library_path(): return ""
def measure_h2d_gbs(*a, **k): raise RuntimeError
EXPORTED_SYMBOLS = []
