# placeholder, replaced below
class ComemError(RuntimeError):
    pass
def _todo(*a, **k):
    raise ComemError("not built yet")
comem_decode_attn = comem_decode_attn_async = comem_decode_attn_host = _todo
comem_decode_attn_workspace_bytes = comem_kv_append_async = comem_status_string = _todo
comem_version = library_path = load_library = _todo
