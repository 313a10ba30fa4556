"""Written by oracle/calibrate_brightness.py (closed-form frame-mean of raw S = 1 at full size)."""
BRIGHTNESS = {
    'C1': 13.827001571655273,
    'C2': 0.005780637729912996,
    'C3': 0.0008480256656184793,
    'C4': 0.005058497190475464,
    'C5': 0.035556189715862274,
}
